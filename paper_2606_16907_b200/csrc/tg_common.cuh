// Shared device/host definitions of libtangram (CUDA side only; the CPU oracle shares nothing
// with this directory).  Notation follows SURVEY.md §8: slice [a,b), island k, mask S, R = S\{k}.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tangram.h"

#define TG_INFU 0x40000000u   // saturating "no plan" (2^30); all DP values are uint32 <= 2^31
#define TG_TINF 0x3fffffffu   // threshold standing for T = infinity: c <= TG_TINF  <=>  c finite
#ifndef TG_NT
#define TG_NT 256             // threads per CTA of the persistent solver
#endif
#ifndef TG_CTAS_PER_SM
#define TG_CTAS_PER_SM 2      // co-resident solver CTAs per SM: each runs its own DP (or its own share of a team's DP), so one
                              // CTA's barriers, copy latencies and level tails are filled by the other
#endif
#define TG_MAX_ITEMS 8192     // (instance, T) DPs per scheduler round
#define TG_QCAP 65536                // queue mode: ring slots (a power of two >= 2 * TG_MAX_ITEMS: round mode uses the first two arrays of it)
#define TG_QUEUE_MAX_INST 1024       // queue mode: at most this many instances; an instance has <= TG_MAX_WISH items in flight, so the
                                     // ring (1024 * 64 = TG_QCAP) cannot wrap onto a live item; the fold checks it anyway (error flag 4)
#define TG_MAX_EVAL 1024      // evaluated thresholds remembered per instance
#define TG_MAX_WISH 64        // DPs per instance and round, upper bound
#define TG_PROBE_FINAL 0x40000000   // flag in probe[]: speculative final DP at the incumbent (S* only; keep every level, back-track)
#define TG_PROBE_KEEP 0x20000000    // flag in probe[]: search probe that also keeps every level and back-tracks (last round of a search)
// item flags: 1 = keep every level and back-track; 2 = the result goes to specOut[item], not out[instance];
//             4 = all islands (a search probe), not only those of the incumbent's mask
#define TG_IT_TRACK 1
#define TG_IT_SPEC 2
#define TG_IT_ALLISL 4
#define TG_CAND_WIN 2048          // candidates staged per instance for the scheduler's bound tests
#define TG_SCHED_SMEM_INST 8      // up to this many instances the scheduler works on shared-memory copies of their search state
#define TG_SPEC_ALL_MAX_INST 4   // up to this many instances every probe of a search's last round back-tracks
#define TG_EDONE 0x40000000   // flag in eIdx: every candidate between the previous evaluated point and this one is resolved
#define TG_KEY_NONE 0xffffffffffffffffull

// Row geometry of the diagonal-major cost tables.  Diagonal d = b - a (1..L).
//   global  cd_k: row d holds a = 0..L-d        (b = a+d <= L),  padded to a multiple of 4
//   staged  Cs_k: row d holds a = 0..L-1-d      (b <= L-1),       padded to a multiple of 4
// tgF(m) = sum_{i=0..m} 4*floor(i/4); sum_{i=0..n} ceil4(i) = tgF(n+3).
__host__ __device__ __forceinline__ uint32_t tgF(int m) {
    if (m < 0) return 0;
    const int q = m >> 2, rem = m & 3;
    return uint32_t(8 * q * (q - 1) + 4 * q * (rem + 1));
}
// offset (words) of global row d (d = 1..L+1): sum_{d'<d} ceil4(L-d'+1)
__host__ __device__ __forceinline__ uint32_t tgGOff(int L, int d) { return tgF(L + 3) - tgF(L - d + 4); }
// offset (words) of staged row d (d = 1..L): sum_{d'<d} ceil4(L-d')
__host__ __device__ __forceinline__ uint32_t tgSOff(int L, int d) { return tgF(L + 2) - tgF(L - d + 3); }

__host__ __device__ __forceinline__ int tgSliceIdx(int L, int a, int b) {
    return a * (2 * L - a + 1) / 2 + (b - a - 1);
}

// Per-instance record in the per-call workspace.  The host fills the pointers and dimensions; the
// loader / prepare kernels fill the derived tables; the solver owns the state block.
struct TgInstDev {
    const int32_t* time_us;  // [NS][K][P] (instance-owned)
    const int32_t* mem_mb;   // [NS][K][P]
    const int32_t* actmem_mb;  // [NS][K][P] MB per in-flight microbatch, or nullptr (NEXT-1: depth-aware memory)
    // NEXT-3(a), tables per signature class (tg_instance_create_classes): the loader reads the class tables
    // (nClasses * K * P entries) instead of the expanded ones; toeplitz = the class of a slice depends on its length only
    // (identical layers): a cost row is then one value per diagonal, kept in cdT and broadcast when the rows are staged
    const int32_t* classOf;    // [NS] class of slice s, or nullptr
    const int32_t* ctime;      // [nClasses][K][P]
    const int32_t* cmem;       // [nClasses][K][P]
    uint32_t* cdT;             // [K][L+2] toeplitz: reduced cost of island k at slice length d (workspace), else nullptr
    int32_t toeplitz;
    const int32_t* slow_us;    // [NS][K][P] slowest internal stage of the partial plan, or nullptr (NEXT-2: multi-stage partial plans)
    uint32_t* thr;             // NEXT-2: [nLayers][K][triG] thresholds of the cells' cost steps (diagonal-major like cd), TG_INFU = no such step
    const int32_t* cap_mb;   // [K]
    const int32_t* bw_gbps;  // [K][K]
    uint32_t* cd;            // [nDepth][K][triG] diagonal-major reduced costs, TG_INFU = none; table q-1 holds the costs
                             // of a stage with q microbatches in flight (q = its own stage + the later ones)
    uint8_t* argp;           // [nDepth][NS][K] lowest p attaining c, 0xff = none
    uint32_t* cand;          // [nCandCap] ascending distinct finite c (first ncand valid)
    uint32_t* sortbuf;       // [NS*K] reduced costs, flat: input of the candidate sort
    uint32_t* sortbuf2;      // [NS*K] scratch of the candidate sort
    uint32_t* sufMin;        // [K][L+2]: sufMin[k][d] = min over d' >= d, b <= L-1 of c  (d = 1..L)
    uint32_t* sufMinAll;     // [K][L+2]: same over all slices (b <= L): longest admissible slice at T
    int32_t* eIdx;           // [TG_MAX_EVAL] evaluated feasible candidates, ascending (bit 30: interval below resolved)
    uint32_t* eF;            // [TG_MAX_EVAL] their f_T
    int32_t L, K, P, m, act_mb, NS, Lp, triG;
    int32_t nDepth;          // 1, or K when actmem_mb is set
    int32_t nLayers;         // 0, or P when slow_us is set: the cost of a cell is then a step function of T -- step j becomes
                             // admissible at thr[j] (ascending in j) and costs cd[j], plan argp[j]; cd / argp hold nLayers tables
    int32_t nTables;         // tables of cd / argp and key sets of the candidate sort: max(nDepth, nLayers, 1)
    int32_t sortCap, ncand;
    uint32_t cminAll[TG_MAX_K];       // min over all slices of c[.][.][k]
    uint32_t maxKey;                  // largest finite reduced cost of any depth (bounds the radix sort's passes)
    long long prepCyc[6];             // TG_DEBUG: clock stamps of the prepare kernel's stages
    const uint32_t* candWin;          // scheduler, few instances: cand[candWinLo .. candWinLo + candWinN) staged in shared memory
    int32_t candWinLo, candWinN;
    int32_t planKind;                 // wide scheduling: item kind returned by this round's planning
    int32_t xbound;                   // NEXT-3(b): transfers are admissible only if x <= T (tg_instance_set_transfer_bound)
    int32_t nAct;                     // NEXT-3(b): 0, or the number of distinct per-boundary activation sizes (tg_instance_set_boundary_act)
    int32_t actVal[TG_MAX_ACT];       // the sizes (MB) by class
    uint32_t* xAct;                   // [nAct][TG_MAX_K * TG_MAX_K] transfer times by size class, sender-major (workspace)
    uint8_t clsOf[256];               // size class of boundary b
    uint32_t x[TG_MAX_K * TG_MAX_K];  // transfer times, sender-major
    // ---- solver state (one scheduler thread per instance) ----
    int32_t phase, loInf, hiFeas, next;   // FEAS bracket: largest infeasible / smallest feasible candidate
    int32_t itemBeg, itemCnt, gstep, nrun;
    int32_t pending;                      // queue mode: items of the current round still running (the CTA that takes it to 0 folds and plans)
    int32_t lbIdx;                        // first candidate passing the necessary condition sum_k maxlen_k(T) >= L
    int32_t incIdx;                       // incumbent = lexicographic min of (iter, candidate index); -1 = none
    int64_t incIter;
    uint32_t incMask;                     // island mask (original labels) of the incumbent's best state
    int32_t nEval, nProbe;
    int32_t specIdx;                      // candidate of a speculative final DP already run (-1 = none)
    int32_t specItem;                     // item of the previous round whose back-tracked result is the incumbent's (-1 = none)
    int32_t probe[TG_MAX_WISH];           // candidates to evaluate this round, ascending
    uint64_t fullWords;  // scratch words of a full-table DP of this instance (K islands alive)
};

enum { TG_PH_NEW = 0, TG_PH_FEAS = 1, TG_PH_BNB = 2, TG_PH_SWEEP = 3, TG_PH_FINAL = 4, TG_PH_DONE = 5 };

// One (instance, T) DP of a scheduler round.
struct TgItem {
    int32_t inst;
    uint32_t T;          // threshold actually applied (TG_TINF for infinity)
    int32_t tidx;        // index into cand, -1 = explicit T (infinity / tg_dp_at)
    uint8_t Ke;          // islands with some admissible slice at T (written by the CTA that runs the item)
    uint8_t flags;       // bit0: keep every level (back-track follows)
    uint8_t isl[TG_MAX_K];  // compact label -> original island
    uint16_t ctaBeg, ctaCnt;  // team of CTAs that runs the item (weighted team mode; written by the scheduler)
    uint32_t seq;        // queue mode: the item's sequence number (the fold checks that its ring slot still holds it)
};

struct TgCtrl {
    int32_t nItems[2];    // per round parity
    uint32_t queue[2];    // solo mode: next item to hand out
    int32_t done;
    int32_t round;
    uint32_t barrier;     // monotone arrival counter of the grid barrier
    int32_t errFlag;
    int32_t nActive;      // instances not done after the previous round's planning (wide scheduling: bounds W)
    // queue mode (a batch of 64..TG_QUEUE_MAX_INST instances): no rounds, the items form one growing queue in a ring
    uint32_t qHead;       // next item sequence number to hand out
    uint32_t qTail;       // next sequence number to reserve for new items
    int32_t nDoneInst;    // instances finished
    int32_t allDone;      // every instance finished: CTAs waiting for an item leave
    int32_t weighted[2];  // per round parity: team sizes follow the items' estimated cost (teamOf / ctaBeg / ctaCnt)
    uint8_t teamOf[2][1024];  // weighted team mode: item of each CTA
    tg_solve_stats stats;
    // debugging aid (TG_DEBUG=1): start time and item count of the first rounds
    unsigned long long roundNs[256];
    int32_t roundItems[256];
    unsigned long long itemNs[8][16];   // team mode: finish time of the first items of the first rounds
    int32_t itemTidx[8][16];
    long long dbgCyc[8][8];
    long long schedCyc[8][4];           // scheduler of the first rounds: clock at entry, after fold, after plan, at exit
};

struct TgSolveCtx {
    TgInstDev* inst;
    int32_t nInst;
    TgItem* items;              // [TG_QCAP]: round mode uses [2][TG_MAX_ITEMS] of it, queue mode the whole ring
    unsigned long long* keys;   // [TG_QCAP], same split: best (value, S, k) per item
    uint32_t* scratch;          // DP tables: nSlots slots of slotWords words
    uint64_t slotWords;         // one slot holds every level of the largest instance of the batch
    int32_t nSlots;             // <= gridDim.x; a slot belongs to one team (team mode) or one CTA (solo mode)
    int32_t wishMax;            // DPs per instance and round, upper bound
    int32_t gallopMax;          // probes of one galloping round
    int32_t wishFloor;          // lower end of the same
    int32_t queueWish;          // queue mode: most probes an instance plans at a time (rounds are cheap there: less speculation pays)
    int32_t wishCap;            // upper end of the per-round probe count chosen from the instance shape (tgWish)
    uint32_t* slotBar;          // [nSlots] arrival counters of the team barriers, zeroed every round
    TgCtrl* ctrl;
    tg_result* specOut;         // [TG_QCAP] results of speculative back-tracks, by item slot
    uint32_t* itemSeq;          // [TG_QCAP] queue mode: sequence number + 1 of the item published in each ring slot
    tg_result* out;
    const uint16_t* rankOf;     // [65536] rank of a mask inside its popcount class
    const uint16_t* maskOf;     // [65536] the inverse: masks ordered by (popcount, value); class r starts at tgPopOff[r]
    uint32_t flags;             // TG_SOLVE_*
    int32_t mode;               // 0 = solve, 1 = single DP at dpT (tg_dp_at)
    uint32_t dpT;
    int32_t dynWords;           // words of dynamic shared memory of a solver CTA
};

// Cost of one cell at threshold T (TG_INFU = no admissible plan); `off` = word offset of the cell inside a [K][triG] table
// (island * triG + row offset + start).  Core / depth tables: the one cost if it is <= T.  NEXT-2 (nLayers > 0): the cost
// of the last step whose threshold is <= T (the thresholds ascend with the step index).  *layer = the step taken.
__device__ __forceinline__ uint32_t tgCostAt(const TgInstDev& I, size_t tableOff, size_t off, uint32_t T, int* layer) {
    if (I.nLayers == 0) {
        if (layer) *layer = 0;
        const uint32_t c = I.cd[tableOff + off];
        return c <= T ? c : TG_INFU;
    }
    const size_t stride = size_t(I.K) * I.triG;
    uint32_t c = TG_INFU;
    for (int j = 0; j < I.nLayers; ++j) {
        if (I.thr[j * stride + off] > T) break;
        c = I.cd[j * stride + off];
        if (layer) *layer = j;
    }
    return c;
}

// The core form alone (the solver's core kernel compiles the step function out).
__device__ __forceinline__ uint32_t tgCostAtCore(const TgInstDev& I, size_t tableOff, size_t off, uint32_t T, int* layer) {
    if (layer) *layer = 0;
    const uint32_t c = I.cd[tableOff + off];
    return c <= T ? c : TG_INFU;
}
__device__ __forceinline__ uint4 tgCostAt4Core(const TgInstDev& I, size_t tableOff, size_t off, uint32_t T) {
    uint4 v = __ldg(reinterpret_cast<const uint4*>(I.cd + tableOff + off));
    v.x = v.x <= T ? v.x : TG_INFU; v.y = v.y <= T ? v.y : TG_INFU;
    v.z = v.z <= T ? v.z : TG_INFU; v.w = v.w <= T ? v.w : TG_INFU;
    return v;
}

// The same for 4 consecutive starts of one row (16-byte aligned offset).
__device__ __forceinline__ uint4 tgCostAt4(const TgInstDev& I, size_t tableOff, size_t off, uint32_t T) {
    if (I.nLayers == 0) {
        uint4 v = __ldg(reinterpret_cast<const uint4*>(I.cd + tableOff + off));
        v.x = v.x <= T ? v.x : TG_INFU; v.y = v.y <= T ? v.y : TG_INFU;
        v.z = v.z <= T ? v.z : TG_INFU; v.w = v.w <= T ? v.w : TG_INFU;
        return v;
    }
    const size_t stride = size_t(I.K) * I.triG;
    uint4 v = make_uint4(TG_INFU, TG_INFU, TG_INFU, TG_INFU);
    for (int j = 0; j < I.nLayers; ++j) {
        const uint4 t = __ldg(reinterpret_cast<const uint4*>(I.thr + j * stride + off));
        if (min(min(t.x, t.y), min(t.z, t.w)) > T) break;
        const uint4 cj = __ldg(reinterpret_cast<const uint4*>(I.cd + j * stride + off));
        v.x = t.x <= T ? cj.x : v.x; v.y = t.y <= T ? cj.y : v.y;
        v.z = t.z <= T ? cj.z : v.z; v.w = t.w <= T ? cj.w : v.w;
    }
    return v;
}

// binomials up to 16 choose r
__constant__ uint16_t tgBinom[17][17];
// start of popcount class r in maskOf: sum_{q<r} C(16, q).  The masks of class r with all bits below Ke are its first
// C(Ke, r) entries (any mask with a higher bit is larger), so one table serves every Ke.
__constant__ uint32_t tgPopOff[18];
