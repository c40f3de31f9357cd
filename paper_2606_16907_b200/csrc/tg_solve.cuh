// Persistent cooperative solver: scheduler state machine, per-T popcount-wavefront DP
// (SURVEY.md §8(a) steps 4-5), threshold-sweep reduction (step 6) and plan back-tracker (step 7).
//
// One launch per tg_solve_batch.  Grid = one CTA of 16 warps per SM (cooperative launch, all co-resident).
// A scheduler round is: CTA 0 folds the previous round's results into the per-instance state
// machines and plans the next list of (instance, T) DPs ("items"); grid barrier; the items are
// executed; grid barrier.  Execution of a round's items:
//   solo mode (items >= slots): every CTA pulls whole DPs from an atomic queue and walks all
//        wavefront levels of its DP alone; levels are separated by __syncthreads only.
//   team mode (items <  slots): the CTAs are dealt to the items in contiguous teams; a team
//        walks the levels of its DP in lockstep, separated by a team barrier (one arrival
//        counter per slot), never by a grid barrier.
// Level r = |R| reads only level r-1 (PAPER.md:250 (2): a stage is added in front of a memoised
// suffix).  State g[a][S][k] is stored as G_r[rank(R)][slot(k)][a], R = S\{k}.
// Inside a level every warp streams over its own range of masks R (see tgWarpLevel).
// This file is compiled TWICE into tg_api.cu (no include guard): namespace tgcore with TG_VAR = 0 -- the core path of
// SURVEY.md §8(a), every variant branch compiled out -- and namespace tgfull with TG_VAR = 1, which also serves the §8(f)
// variants (footprint tables, multi-stage partial plans, per-boundary activation sizes).  The host launches tgfull only
// when an instance of the batch uses one of them: the variants' extra template instances and branches measurably slowed
// the core workloads (cfg5 +3.7 %, cfg4 +1.6 %) when they shared one kernel.
#include "tg_common.cuh"
#include "tg_prep.cuh"
#if !defined(TG_SOLVE_NS) || !defined(TG_VAR)
#error "define TG_SOLVE_NS and TG_VAR before including tg_solve.cuh"
#endif
#define TG_COST_AT(I, tableOff, off, T, layer) (TG_VAR ? tgCostAt((I), tableOff, off, T, layer) : tgCostAtCore((I), tableOff, off, T, layer))
#define TG_COST_AT4(I, tableOff, off, T) (TG_VAR ? tgCostAt4((I), tableOff, off, T) : tgCostAt4Core((I), tableOff, off, T))

#define TG_NW (TG_NT / 32)     // warps per CTA
#ifndef TG_STAGE_TMA
#define TG_STAGE_TMA 0          // 1: stage the cost rows with TMA bulk copies (A/B variant, see tgStageCosts)
#endif
#define TG_NB_MAX 256   // masks per batch, upper bound (row index inside a batch fits 16 bits: 256 * 16)
#define TG_DESC_W 6     // words of a mask descriptor: R | cap(R) << 16, pad, non-members (16 nibbles), members (16 nibbles)

namespace TG_SOLVE_NS {

struct TgShared {
    // staged item
    int useGlobalC;
    int sL, sLp, sKe, sInst;
    uint32_t sT;
    // row windows (see "Row windows" below): rows hold Wd starts, row of state (S, k) begins at start lo4(cap(S))
    int sWd, sSlack, sWindowed;
    // split of the dynamic shared memory for this item: [cost rows | batch buffers of the level (tgLevelBatched)]
    int batchOff;
    int nWarps, wbufWords, wbufOff;   // team mode: [cost rows | nWarps x wbufWords of warp-private row buffers]
    uint32_t rowOf[TG_NW][2 * TG_MAX_K];   // team mode: source row of each member of the mask being issued (per half warp)
    uint8_t kl[TG_NW][2 * TG_MAX_K];       // team mode: islands not in the current mask, ascending (per half warp)
    int cntP[2][TG_MAX_K];          // rows of each island in a batch, counted by its prepass (per batch parity)
    int cur[2][TG_MAX_K];           // next free list position of each island (starts at the prefix of the counts)
    int csUsed4;                    // 16-byte words of the staged cost rows of all islands (incl. the pads between them)
    uint32_t cdOff;                 // word offset of the reduced table of the depth currently staged
    uint8_t maxlenK[TG_MAX_K];      // longest admissible slice of island k at T, any position
    uint16_t capLo[256], capHi[256];   // cap(R) = capLo[R & 255] + capHi[R >> 8]: sums of maxlenK over the low / high islands of a mask
    uint32_t baseK[TG_MAX_K];
    int dmaxK[TG_MAX_K];
    uint8_t dmaxTile[TG_MAX_K][64];
    alignas(16) uint32_t xS[TG_MAX_K][TG_MAX_K];
    alignas(16) uint32_t xInf[TG_MAX_K];            // all-INF transfer row for a lane's unused k slot
    int sNAct;                      // per-boundary activation sizes (NEXT-3(b)): number of size classes, 0 = one scalar size
    int xOff;                       // their transfer matrices [sNAct][TG_MAX_K][TG_MAX_K] sit in the dynamic shared memory at this word
    uint8_t clsOfS[256];            // size class of boundary b
    uint8_t isl[TG_MAX_K];
    uint16_t binom[17][17];
    // scheduler / queue
    uint32_t warpSums[33];
    float wgt[32];                  // estimated cost of the round's items (weighted team mode)
    int iTmp[8];
    unsigned long long llTmp[2];
    int curItem;
#if TG_STAGE_TMA
    alignas(8) unsigned long long mbar;   // completion barrier of the bulk copies of the cost rows
    uint32_t mbarPhase;
#endif
    long long tmark;                // phase timer of thread 0
    unsigned long long cyc[8];      // per-CTA cycle counters, flushed to the statistics at exit
};

__device__ __forceinline__ uint32_t tgSmemAddr(const void* p) { return uint32_t(__cvta_generic_to_shared(p)); }

// Phase timer: thread 0 charges the cycles since its previous mark to counter `which`.
__device__ __forceinline__ void tgMark(TgShared& sm, int which) {
    if (threadIdx.x == 0) {
        const long long now = clock64();
        sm.cyc[which] += (unsigned long long)(now - sm.tmark);
        sm.tmark = now;
    }
}

__device__ __forceinline__ uint32_t tgAddMin(uint32_t a, uint32_t b, uint32_t c) { return __viaddmin_u32(a, b, c); }

// Grid-wide barrier on a monotone counter (all CTAs are co-resident: cooperative launch).
__device__ __forceinline__ void tgGridBarrier(TgCtrl* ctrl, uint32_t& epoch) {
    __syncthreads();
    if (threadIdx.x == 0) {
        ++epoch;
        const uint32_t target = epoch * gridDim.x;
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(&ctrl->barrier) : "memory");
        while (true) {
            uint32_t v;
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(&ctrl->barrier) : "memory");
            if (int32_t(v - target) >= 0) break;
            __nanosleep(32);
        }
    }
    __syncthreads();
}

// Barrier of one team on its slot counter (zeroed by the scheduler every round).
__device__ __forceinline__ void tgTeamBarrier(uint32_t* bar, uint32_t target) {
    __syncthreads();
    if (threadIdx.x == 0) {
        // release-arrive / acquire-poll: the CTA's writes (ordered before this thread by the barrier above) become
        // visible to whoever observes the count, and what the other members wrote is visible after the poll
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar) : "memory");
        uint32_t v;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
        } while (v < target);
    }
    __syncthreads();
}

// The same barrier in two halves: arrive when the level is done, wait at the start of the next level -- behind the table
// look-ups of that level's first masks, which need nothing the other members write (tgRunItem).
__device__ __forceinline__ void tgTeamArrive(uint32_t* bar) {
    __syncthreads();
    if (threadIdx.x == 0) asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar) : "memory");
}
__device__ __forceinline__ void tgTeamWait(uint32_t* bar, uint32_t target) {
    if (threadIdx.x == 0) {
        uint32_t v;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
        } while (v < target);
    }
    __syncthreads();
}

// rows (R,k) of wavefront level r with Ke islands alive
__device__ __forceinline__ uint32_t tgLevelRows(int Ke, int r) { return uint32_t(tgBinom[Ke][r]) * uint32_t(Ke - r); }

// word offset of level r inside a slot: ping-pong halves, or every level kept (bufWords == 0)
__device__ __forceinline__ uint64_t tgLevelOff(uint64_t bufWords, int Ke, int Lp, int r) {
    if (bufWords) return uint64_t(r & 1) * bufWords;
    uint64_t rows = 0;
    for (int q = 0; q < r; ++q) rows += tgLevelRows(Ke, q);
    return rows * uint64_t(Lp);
}

// Row windows.  With maxlen_k = longest admissible slice of island k at T and cap(S) = sum of maxlen
// over S, a state (a, S, k) is finite only if L - a <= cap(S), and it can be part of a full plan
// only if the prefix [0, a) fits the other islands: a <= Ctot - cap(S), Ctot = cap(all).  So every
// row needs just the starts  a in [L - cap(S), Ctot - cap(S)]  — Ctot - L + 1 of them, usually a small
// fraction of L near T*.  Rows are stored with Wd = ceil4(Ctot - L + 4) entries beginning at the
// 4-aligned start lo4(S) = floor4(max(0, L - cap(S))); entries left of the window are INF by the
// first bound, entries right of it are never read by a state inside its own window.
__device__ __forceinline__ int tgLo4(const TgShared& sm, int cap) {
    return sm.sWindowed ? (max(0, sm.sL - cap) & ~3) : 0;
}

// division of small numbers by a CTA-uniform divisor d: q = t / d for t * d < 2^32 (magic = ceil(2^32 / d), 0 for d = 1)
// (divisors up to 32 -- chunks of a row window, row groups of a mask -- come from a constant table: a 32-bit division is a
// dependent chain of ~70 instructions, and the level geometry below sits on every level's critical path)
__constant__ uint32_t tgMagicTab[33] = {0u, 0u, 2147483648u, 1431655766u, 1073741824u, 858993460u, 715827883u, 613566757u, 536870912u, 477218589u, 429496730u, 390451573u, 357913942u, 330382100u, 306783379u, 286331154u, 268435456u, 252645136u, 238609295u, 226050911u, 214748365u, 204522253u, 195225787u, 186737709u, 178956971u, 171798692u, 165191050u, 159072863u, 153391690u, 148102321u, 143165577u, 138547333u, 134217728u};
__device__ __forceinline__ uint32_t tgMagic(uint32_t d) { return d <= 32u ? tgMagicTab[d] : 0xffffffffu / d + 1u; }
__device__ __forceinline__ uint32_t tgDivM(uint32_t t, uint32_t magic) { return magic ? __umulhi(t, magic) : t; }

// Fills the staged cost rows (and dmaxTile) from the reduced table of depth q (q = 1 unless the instance has
// an actmem table: then level r of the DP, whose stages have r later stages, uses q = r + 1 -- SURVEY NEXT-1).
// The layout (baseK, D_k) comes from depth 1, whose costs are the lowest, so it covers every depth.
// Returns this thread's count of admissible entries; ends with a CTA barrier.
__device__ unsigned tgStageCosts(const TgSolveCtx& ctx, TgShared& sm, uint32_t* Cs, int q, bool count) {
    const int tid = threadIdx.x;
    const TgInstDev& I = ctx.inst[sm.sInst];
    const int L = sm.sL, Lp = sm.sLp, Ke = sm.sKe, nb4 = Lp >> 2;
    const uint32_t T = sm.sT;
    unsigned nAdm = 0;
    if (tid == 0) sm.cdOff = uint32_t(q - 1) * uint32_t(I.K) * uint32_t(I.triG);
    __syncthreads();
    if (!sm.useGlobalC) {
        // one flat loop over the 16-byte words of every island's rows (island k occupies D_k * nb4 + 1 of them from
        // baseK[k] / 4): all loads of a thread are independent, one trip to L2 for the whole table instead of one
        // per island
#if TG_STAGE_TMA
        // A/B variant (profiles/r2_sass_summary.md): the raw cost rows come in as TMA bulk copies (cp.async.bulk, one per
        // island and diagonal, completion on an mbarrier) and are thresholded in place; core tables only.
        const bool bulk = !(TG_VAR && I.nLayers);
        if (bulk) {
            const uint32_t mbar = tgSmemAddr(&sm.mbar);
            const uint32_t phase = sm.mbarPhase;
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // earlier generic-proxy writes of this memory are ordered first
            uint32_t bytes = 0;
            int rows = 0;
            for (int kc = 0; kc < Ke; ++kc) rows += sm.dmaxK[kc];
            for (int rw = tid; rw < rows; rw += TG_NT) {
                int kc = 0, d = rw;
                while (d >= sm.dmaxK[kc]) { d -= sm.dmaxK[kc]; ++kc; }
                ++d;
                const uint32_t words = uint32_t(min(Lp, (L - d + 1 + 3) & ~3));
                const uint32_t* src = I.cd + sm.cdOff + size_t(sm.isl[kc]) * I.triG + tgGOff(L, d);
                const uint32_t dst = tgSmemAddr(Cs + sm.baseK[kc] + (d - 1) * Lp);
                asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                             ::"r"(dst), "l"(src), "r"(words * 4u), "r"(mbar) : "memory");
                bytes += words * 4u;
            }
            if (bytes) asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
            else asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mbar) : "memory");
            uint32_t done = 0;
            while (!done)
                asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                             : "=r"(done) : "r"(mbar), "r"(phase) : "memory");
        }
#else
        const bool bulk = false;
#endif
        // A thread takes one column (island, 4 starts) -- or one of S interleaved shares of its diagonals when there are fewer
        // columns than threads -- and walks down the diagonals: island, start and base addresses are worked out once per
        // column, a step is a load, the threshold, the row-end mask and a store.  (The flat loop over the 16-byte words that
        // was here spent ~125 instructions a word on finding its island and diagonal: 12-15k of an item's 22-26k staging
        // cycles at cfg3 / cfg4 were instruction issue.)  Four loads of a thread are in flight.
        const uint32_t mNb4 = tgMagic(uint32_t(nb4));
        const uint32_t* const cdP = I.cd + sm.cdOff;
        const uint32_t* const cdTP = I.cdT;
        const size_t triG = size_t(I.triG);
        const bool layered = TG_VAR && I.nLayers != 0;
        const int nCols = Ke * nb4;
        int sh = 0;
        while (sh < 3 && (nCols << (sh + 1)) <= TG_NT) ++sh;   // S = 2^sh threads a column
        const int S = 1 << sh;
        for (int cs0 = 0; cs0 < (nCols << sh); cs0 += TG_NT) {   // (warp-uniform trips: the shares of a column meet in a shuffle below)
            const int cs = cs0 + tid;
            const bool active = cs < (nCols << sh);
            const int col = active ? (cs >> sh) : 0, sub = cs & (S - 1);
            const int kc = int(tgDivM(uint32_t(col), mNb4)), a4 = col - kc * nb4, a = 4 * a4;
            const int dk = active ? sm.dmaxK[kc] : 0, Dk = (dk + 3) & ~3;
            int dTop = 0;   // widest diagonal of this share with an admissible entry
            uint4* const dst = reinterpret_cast<uint4*>(Cs + sm.baseK[kc]) + a4;
            const size_t islOff = size_t(sm.isl[kc]) * triG + size_t(a);
            const int islT = int(sm.isl[kc]) * (L + 2);
            for (int d0 = 1 + sub; d0 <= Dk; d0 += 4 * S) {
                uint4 v[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int d = d0 + u * S;
                    v[u] = make_uint4(TG_INFU, TG_INFU, TG_INFU, TG_INFU);
                    if (d <= dk && a4 < ((L - d + 3) >> 2)) {
                        if (bulk) {
                            v[u] = dst[(d - 1) * nb4];
                        } else if (cdTP) {
                            // identical layers (NEXT-3(a)): the row is one value, read once per diagonal instead of once per start
                            const uint32_t cv = __ldg(cdTP + islT + d);
                            v[u] = make_uint4(cv, cv, cv, cv);
                        } else if (layered) {
                            v[u] = TG_COST_AT4(I, sm.cdOff, islOff + tgGOff(L, d), T);
                        } else {
                            v[u] = __ldg(reinterpret_cast<const uint4*>(cdP + islOff + tgGOff(L, d)));
                        }
                    }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int d = d0 + u * S;
                    if (d > Dk) continue;
                    const int amax = L - 1 - d;
                    uint4 x = v[u];
                    // (multi-stage partial plans, NEXT-2: admissible by the slowest internal stage, already applied by
                    // TG_COST_AT4 -- the cost itself, the whole time, may exceed T)
                    const uint32_t Tc = layered ? TG_INFU - 1u : T;
                    x.x = (x.x <= Tc && a + 0 <= amax) ? x.x : TG_INFU;
                    x.y = (x.y <= Tc && a + 1 <= amax) ? x.y : TG_INFU;
                    x.z = (x.z <= Tc && a + 2 <= amax) ? x.z : TG_INFU;
                    x.w = (x.w <= Tc && a + 3 <= amax) ? x.w : TG_INFU;
                    const unsigned fin = (x.x < TG_INFU) + (x.y < TG_INFU) + (x.z < TG_INFU) + (x.w < TG_INFU);
                    nAdm += fin;
                    if (fin) dTop = max(dTop, d);
                    dst[(d - 1) * nb4] = x;
                }
            }
            // dmaxTile = widest admissible diagonal of the column's 4 starts (bounds the phase-2 loop): the column's S shares
            // are neighbouring lanes
            for (int o = 1; o < S; o <<= 1) dTop = max(dTop, __shfl_xor_sync(0xffffffffu, dTop, o));
            if (active && sub == 0) sm.dmaxTile[kc][a4] = uint8_t(dTop);
        }
#if TG_STAGE_TMA
        __syncthreads();
        if (bulk && tid == 0) sm.mbarPhase ^= 1u;
#endif
    } else {
        for (int w = tid; w < Ke * nb4; w += TG_NT) {
            const int kc = w / nb4, a4 = w - kc * nb4;
            sm.dmaxTile[kc][a4] = uint8_t(max(0, min(sm.dmaxK[kc], L - 1 - 4 * a4)));
        }
        if (count)
            for (int kc = 0; kc < Ke; ++kc) {
                const uint32_t* cdk = ((TG_VAR && I.nLayers) ? I.thr : I.cd + sm.cdOff) + size_t(sm.isl[kc]) * I.triG;   // (NEXT-2: admissible from the first step on)
                for (int d = 1; d <= sm.dmaxK[kc]; ++d)
                    for (int a = tid; a <= L - 1 - d; a += TG_NT) nAdm += cdk[tgGOff(L, d) + a] <= T ? 1u : 0u;
            }
    }
    __syncthreads();
    return nAdm;
}

// words between consecutive rows of a warp's buffer: 4 (mod 8), so consecutive rows start in different 16-byte
// bank groups (rows are read by several island groups at the same chunk offset)
__device__ __forceinline__ int tgRowStride(int Wd) { return Wd + 12 + (((Wd + 12) & 7) == 0 ? 4 : 0); }
// words between consecutive source rows in shared memory: a multiple of 4 with an odd number of 16-byte
// units, so rows of neighbouring masks start in different bank groups
__device__ __forceinline__ int tgSrcStride(int Wd) { return Wd + 4 + (((Wd + 4) & 7) == 0 ? 4 : 0); }

// ---------------------------------------------------------------------------------------------
// Staging of one item's thresholded cost tables into shared memory.
//   Cs_k[(d-1)*Lp + a] = c[a][a+d][k] if <= T and a+d <= L-1, else INF   (k in compact labels)
// Rows d = 1..D_k, D_k = dmaxK[k] (widest admissible slice of island k at T) rounded up to a
// multiple of 4 so that the min-plus loop needs no row predicate; uniform row stride Lp.
// dmaxTile[k][t] = widest admissible diagonal of starts a = 4t..4t+3: bounds the phase-2 loop.
// ---------------------------------------------------------------------------------------------
__device__ void tgStageItem(const TgSolveCtx& ctx, TgShared& sm, uint32_t* Cs, uint32_t*, const TgItem* itp, bool count, bool team) {
    __syncthreads();
    unsigned nAdm = 0;   // admissible (a, b, k) cost entries with b <= L-1 seen by this thread
    const int tid = threadIdx.x, lane = tid & 31;
    const TgInstDev& I = ctx.inst[__ldcg(&itp->inst)];
    const int L = I.L, Lp = I.Lp;
    const uint32_t T = __ldcg(&itp->T);
    // geometry of the item: the islands with some admissible slice at T, in compact labels.  The final
    // DP only needs the islands of the optimal mask S*: S* is the lowest mask attaining the optimum at
    // T*, so no subset of it ties, and the back-track never leaves its subsets.
    if (tid < 32) {
        const int fl = __ldcg(&itp->flags);
        const uint32_t allow = ((fl & TG_IT_TRACK) && !(fl & TG_IT_ALLISL) && ctx.mode == 0) ? I.incMask : 0xffffu;
        const bool ok = lane < I.K && I.cminAll[lane] <= T && (allow >> lane & 1u);
        const uint32_t bal = __ballot_sync(0xffffffffu, ok);
        if (lane < TG_MAX_K) sm.isl[lane] = 0;
        __syncwarp();
        if (ok) sm.isl[__popc(bal & ((1u << lane) - 1u))] = uint8_t(lane);
        if (lane == 0) { sm.sL = L; sm.sLp = Lp; sm.sKe = __popc(bal); sm.sT = T; sm.sInst = __ldcg(&itp->inst); }
    }
    __syncthreads();
    const int Ke = sm.sKe;
    if (count) {   // member 0 publishes the geometry (the scheduler maps the best state's mask back through isl) and counts
        TgItem* itw = const_cast<TgItem*>(itp);
        if (tid < TG_MAX_K) itw->isl[tid] = sm.isl[tid];
        if (tid == 0) {
            itw->Ke = uint8_t(Ke);
            atomicAdd((unsigned long long*)&ctx.ctrl->stats.plans_dense, (unsigned long long)I.NS * I.K << (I.K - 1));
            if (Ke) atomicAdd((unsigned long long*)&ctx.ctrl->stats.states_live, (unsigned long long)L * Ke << (Ke - 1));
        }
    }
    for (int w = tid; w < Ke * Ke; w += TG_NT) {
        const int kc = w / Ke, jc = w - kc * Ke;
        const uint32_t xv = I.x[int(sm.isl[kc]) * TG_MAX_K + int(sm.isl[jc])];
        sm.xS[kc][jc] = (I.xbound && xv > T) ? TG_INFU : xv;   // transfer bound (NEXT-3(b)): a slower link is not admissible at T
    }
    if (TG_VAR && I.nAct) for (int w = tid; w < 256; w += TG_NT) sm.clsOfS[w] = I.clsOf[w];
    if (tid == 0) sm.sNAct = TG_VAR ? I.nAct : 0;
    // widest diagonal with an admissible entry (b <= L-1) and longest admissible slice at any position (b <= L) of
    // every island: sufMin / sufMinAll are non-decreasing in d, so each is the number of lengths whose entry is
    // <= T.  One warp per island, lanes over the lengths: one round trip to L2 instead of a binary search's seven.
    {
        for (int w = tid >> 5; w < Ke; w += TG_NW) {
            const uint32_t* sf = I.sufMin + size_t(sm.isl[w]) * (L + 2);
            const uint32_t* sa = I.sufMinAll + size_t(sm.isl[w]) * (L + 2);
            unsigned nd = 0, nl = 0;
            for (int d0 = 1 + lane; d0 <= L; d0 += 64) {   // two lengths a lane and trip, their four loads issued together
                const int d1 = d0 + 32;
                const uint32_t f0 = sf[d0], a0 = sa[d0];
                const uint32_t f1 = d1 <= L ? sf[d1] : TG_INFU, a1 = d1 <= L ? sa[d1] : TG_INFU;
                nd += ((d0 <= L - 1 && f0 <= T) ? 1u : 0u) + ((d1 <= L - 1 && f1 <= T) ? 1u : 0u);
                nl += ((a0 <= T) ? 1u : 0u) + ((d1 <= L && a1 <= T) ? 1u : 0u);
            }
            nd = __reduce_add_sync(0xffffffffu, nd);
            nl = __reduce_add_sync(0xffffffffu, nl);
            if (lane == 0) { sm.dmaxK[w] = int(nd); sm.maxlenK[w] = uint8_t(nl); }
        }
    }
    __syncthreads();
    for (int t = tid; t < 256; t += TG_NT) {   // cap(R) by two look-ups instead of a reduction over the members of every mask
        int lo = 0, hi = 0;
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            if ((t >> e & 1) && e < Ke) lo += sm.maxlenK[e];
            if ((t >> e & 1) && 8 + e < Ke) hi += sm.maxlenK[8 + e];
        }
        sm.capLo[t] = uint16_t(lo); sm.capHi[t] = uint16_t(hi);
    }
    if (tid == 0) {
        int ctot = 0;
        for (int kc = 0; kc < Ke; ++kc) ctot += sm.maxlenK[kc];
        const int wd = (ctot - L + 4 + 3) & ~3;
        sm.sSlack = ctot - L;
        sm.sWindowed = (ctot >= L && wd < Lp) ? 1 : 0;
        sm.sWd = sm.sWindowed ? wd : Lp;
        uint32_t acc = 0;
        // + 4 words per island: tables of different islands start in different 16-byte bank groups, so the
        // island groups of a warp do not collide when they read the same diagonal
        for (int kc = 0; kc < Ke; ++kc) { sm.baseK[kc] = acc; acc += uint32_t((sm.dmaxK[kc] + 3) & ~3) * uint32_t(Lp) + 4u; }
        // dynamic shared memory of this item: the cost rows if a batch of at least 8 masks still fits behind them
        // at the level that needs the most rows per mask (else the L2 fallback), the rest for the batches
        const int HS = tgRowStride(sm.sWd), SS = tgSrcStride(sm.sWd);
        int perMask = 0;
        for (int r = 1; r < Ke; ++r) perMask = max(perMask, (Ke - r) * HS + 2 * r * SS);
        perMask += 2 * TG_DESC_W + 4 * Ke;
        const int xWords = TG_VAR ? I.nAct * TG_MAX_K * TG_MAX_K : 0;      // transfer matrices of the activation-size classes (NEXT-3(b))
        sm.useGlobalC = int64_t(acc) + xWords + 16 + 8ll * perMask > int64_t(ctx.dynWords) ? 1 : 0;
        sm.csUsed4 = int(acc >> 2);
        sm.xOff = sm.useGlobalC ? 0 : int((acc + 3u) & ~3u);
        sm.batchOff = sm.xOff + xWords;
        if (team) {
            // team mode: every warp gets room for one mask's rows at the widest level (2 Ke - 1 rows), the cost rows come
            // next if they still fit, and what is left doubles the warps' buffers so that two masks run side by side
            const int total = ctx.dynWords - xWords;
            const int perMaskW = max(1, 2 * Ke - 1) * HS;
            const int nWp = max(1, min(TG_NW, total / perMaskW));
            sm.useGlobalC = acc > uint32_t(total - nWp * perMaskW) ? 1 : 0;
            const int csUsed = sm.useGlobalC ? 0 : int((acc + 3u) & ~3u);
            sm.nWarps = nWp;
            sm.xOff = csUsed;
            sm.wbufOff = csUsed + xWords;
            sm.wbufWords = min(2 * perMaskW, (total - csUsed) / nWp) & ~3;
        }
        if (count) {
            if (sm.useGlobalC) atomicAdd((unsigned long long*)&ctx.ctrl->stats.n_items_global_c, 1ull);
            if (Ke && sm.sSlack >= 0) atomicAdd((unsigned long long*)&ctx.ctrl->stats.states_windowed, (unsigned long long)sm.sWd * Ke << (Ke - 1));
        }
    }
    __syncthreads();
    if (TG_VAR && I.nAct) {   // the transfer matrices of the size classes, thresholded like xS
        uint32_t* xd = Cs + sm.xOff;
        for (int w = tid; w < I.nAct * Ke * Ke; w += TG_NT) {
            const int cls = w / (Ke * Ke), e = w - cls * Ke * Ke, kc = e / Ke, jc = e - kc * Ke;
            const uint32_t xv = I.xAct[cls * (TG_MAX_K * TG_MAX_K) + int(sm.isl[kc]) * TG_MAX_K + int(sm.isl[jc])];
            xd[cls * (TG_MAX_K * TG_MAX_K) + kc * TG_MAX_K + jc] = (I.xbound && xv > T) ? TG_INFU : xv;
        }
    }
    nAdm = tgStageCosts(ctx, sm, Cs, 1, count);
    if (count) {   // statistics: admissible relaxations of this DP (stage + transfer)
        for (int o = 16; o > 0; o >>= 1) nAdm += __shfl_down_sync(0xffffffffu, nAdm, o);
        if (lane == 0 && nAdm && Ke > 0)
            atomicAdd((unsigned long long*)&ctx.ctrl->stats.relax_admissible, (unsigned long long)nAdm << (Ke - 1));
        if (tid == 0 && Ke >= 2)
            atomicAdd((unsigned long long*)&ctx.ctrl->stats.relax_admissible, (unsigned long long)L * Ke * (Ke - 1) << (Ke - 2));
    }
    __syncthreads();
}

// ---------------------------------------------------------------------------------------------
// Level 0: R = {} : G_0[k][a] = c[a][L][k] if <= T  (single stage [a,L) on island k)
// Every member of a team writes the same values (saves one team barrier); member 0 posts the key.
// ---------------------------------------------------------------------------------------------
__device__ void tgLevel0(const TgSolveCtx& ctx, TgShared& sm, uint32_t* G, unsigned long long* key, bool post) {
    const TgInstDev& I = ctx.inst[sm.sInst];
    const int L = sm.sL, Wd = sm.sWd, Ke = sm.sKe;
    const uint32_t T = sm.sT;
    for (int w = threadIdx.x; w < Ke * Wd; w += TG_NT) {
        const int kc = w / Wd, a = tgLo4(sm, sm.maxlenK[kc]) + (w - kc * Wd);
        uint32_t v = TG_INFU;
        if (a < L) {
            v = TG_COST_AT(I, 0, size_t(sm.isl[kc]) * I.triG + tgGOff(L, L - a) + a, T, nullptr);
        }
        G[w] = v;
        if (post && a == 0 && v < TG_INFU)
            atomicMin(key, (unsigned long long)v << 32 | (unsigned long long)(1u << kc) << 8 | (unsigned long long)kc);
    }
}

// ---------------------------------------------------------------------------------------------
// Levels r >= 1: the CTA walks its share of the level's masks in BATCHES of NB masks (colexicographic
// rank order).  Per batch, all threads of the CTA:
//   prepass  (one thread per mask, one batch ahead)  mask R from its rank (table maskOf), cap(R) and the
//            nibble lists of its members / non-members -> a 6-word descriptor in shared memory
//   copies   16-byte cp.async (LDGSTS) of the batch's r source rows G_{r-1}[R\{j}][j][.] per mask into shared
//            memory, one batch ahead of their use (double buffer); source row = rankOf[R\{j}] (table)
//   phase 1  H[R][k][b] = min_{j in R} x[k][j] + src[j][b]          item = (mask, 4 consecutive b, NSL rows k)
//            and, per row (R, k), an 8-byte row record appended to the list of island k
//   phase 2  G_r[R][k][a] = min_{b>a} Cs_k[a][b] + H[R][k][b]       item = (row, 4 consecutive a), rows taken
//            ISLAND BY ISLAND from the lists: the lanes of a warp then share the cost table of one island and
//            run (nearly) the same number of diagonal blocks.  (Round 1 gave one warp one mask: its rows
//            belong to different islands whose admissible diagonals differ by up to 19:1, and the ncu source
//            page showed 10-14 of 32 lanes active in the min-plus loop.)
// Two CTA barriers per batch.  Shared memory of a batch: [descriptors x2 | lists | H rows | source rows x2].
// ---------------------------------------------------------------------------------------------


__device__ __forceinline__ uint4 tgLds4(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint32_t tgLds1(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void tgSts4(uint32_t addr, uint4 v) {
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}


// prepass of one mask: descriptor from the mask's rank inside level r, the rows of its r sources in level r-1 and one
// count per non-member island (the island lists of phase 2 are laid out from these counts).
// Source row of member j of R = state (R\{j}, first island j): mask rank from the table, slot of j among the
// non-members of R\{j} = j - (members of R below j).
__device__ __forceinline__ void tgPrepassMask(const TgSolveCtx& ctx, const TgShared& sm, uint32_t* desc, uint32_t* srcRow, int* cntP,
                                              uint32_t rank, int r, int Ke) {
    const uint32_t R = __ldg(ctx.maskOf + tgPopOff[r] + rank);
    uint32_t klLo = 0, klHi = 0;
    int nm = 0, nc = 0;
    const int nk = Ke - r;
    // the rank look-ups of all islands are issued together (a non-member's look-up is a valid, unused table entry): one
    // load latency on the level's critical path instead of r
    uint16_t rk[TG_MAX_K];
#pragma unroll
    for (int e = 0; e < TG_MAX_K; ++e) rk[e] = e < Ke ? __ldg(ctx.rankOf + (R ^ (1u << e))) : uint16_t(0);
#pragma unroll
    for (int e = 0; e < TG_MAX_K; ++e) {
        if (e >= Ke) break;
        if (R >> e & 1u) {
            srcRow[nm] = uint32_t(rk[e]) * uint32_t(nk + 1) + uint32_t(e - nm);
            ++nm;
        } else {
            if (nc < 8) klLo |= uint32_t(e) << (4 * nc); else klHi |= uint32_t(e) << (4 * (nc - 8));
            ++nc;
            atomicAdd(&cntP[e], 1);
        }
    }
    desc[0] = R | (uint32_t(sm.capLo[R & 255u]) + uint32_t(sm.capHi[R >> 8])) << 16;
    desc[2] = klLo; desc[3] = klHi;
}

__device__ __forceinline__ uint32_t tgNibble(uint32_t lo, uint32_t hi, int i) { return ((i < 8 ? lo : hi) >> (4 * (i & 7))) & 15u; }

// copies of a batch's source rows: item = (source row pr = i * r + ji of the batch, chunk of 4 starts), chunk fastest
// (coalesced 16-byte pieces); the row's index in level r-1 was looked up by the prepass.
__device__ __forceinline__ void tgIssueBatch(const uint32_t* srcRow, uint32_t srcAddr, const uint32_t* Gprev, int nb, int r, int Wd,
                                             int nbw, uint32_t mNbw, uint32_t SSB) {
    const int nItems = nb * r * nbw;
    for (int t = threadIdx.x; t < nItems; t += TG_NT) {
        const uint32_t pr = tgDivM(uint32_t(t), mNbw), ch = uint32_t(t) - pr * uint32_t(nbw);
        const uint32_t* src = Gprev + size_t(srcRow[pr]) * Wd + 4u * ch;
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(srcAddr + pr * SSB + ch * 16u), "l"(src) : "memory");
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
}

#define TG_SPL 8   // most k slots (rows) a phase-1 item handles together (accumulators: TG_SPL x 4)

// phase 1 of a batch.  Item = (mask i, chunk ch of 4 consecutive b, group sg of NSL rows): the chunk of every
// source row is read once (LDS.128) and serves NSL rows; slots past the mask's last row read an all-INF x row.
// (The island lists phase 2 works from are filed by tgBuildLists below, during the same phase.)
template <int NSL, bool ACTB>
__device__ __forceinline__ void tgPhase1B(const TgShared& sm, const uint32_t* desc, uint32_t srcAddr, uint32_t hAddr,
                                          int nb, int r, int nk, int nbw, int nsg, uint32_t mNbw, uint32_t mNsg, uint32_t SSB,
                                          uint32_t HSB, uint32_t xsBase, uint32_t xInfAddr) {
    const int nItems = nb * nbw * nsg;
    const int Lw = sm.sWindowed ? sm.sL : 0;
    for (int t = threadIdx.x; t < nItems; t += TG_NT) {
        const uint32_t u = tgDivM(uint32_t(t), mNbw), ch = uint32_t(t) - u * uint32_t(nbw);
        const uint32_t i = tgDivM(u, mNsg), sg = u - i * uint32_t(nsg);
        const uint32_t* d = desc + i * TG_DESC_W;
        const uint32_t w0 = d[0], klLo = d[2], klHi = d[3];
        const uint32_t R = w0 & 0xffffu;
        const int s0 = int(sg) * NSL;
        uint32_t xrow[NSL];
#pragma unroll
        for (int e = 0; e < NSL; ++e)
            xrow[e] = (s0 + e < nk) ? xsBase + tgNibble(klLo, klHi, s0 + e) * (TG_MAX_K * 4u) : xInfAddr;
        uint32_t acc[NSL][4];
#pragma unroll
        for (int e = 0; e < NSL; ++e) { acc[e][0] = acc[e][1] = acc[e][2] = acc[e][3] = TG_INFU; }
        uint32_t sA = srcAddr + i * uint32_t(r) * SSB + ch * 16u;
        uint32_t Rb = R;
        uint32_t co[4] = {0, 0, 0, 0};   // ACTB: byte offset of the transfer matrix of each of the chunk's 4 boundaries
        if (ACTB) {
            const int b0 = (max(0, Lw - int(w0 >> 16)) & ~3) + 4 * int(ch);   // the H row starts at b = lo4(R)
#pragma unroll
            for (int cq = 0; cq < 4; ++cq) co[cq] = uint32_t(sm.clsOfS[min(b0 + cq, 255)]) * (TG_MAX_K * TG_MAX_K * 4u);
        }
#pragma unroll 2
        for (int ji = 0; ji < r; ++ji) {
            const uint32_t j4 = uint32_t(__ffs(Rb) - 1) * 4u;
            Rb &= Rb - 1;
            const uint4 g4 = tgLds4(sA);
            sA += SSB;
#pragma unroll
            for (int e = 0; e < NSL; ++e) {
                if (ACTB) {
                    const bool ok = s0 + e < nk;                 // (an unused slot reads the one all-INF row)
                    const uint32_t xa = xrow[e] + j4;
                    acc[e][0] = tgAddMin(tgLds1(xa + (ok ? co[0] : 0u)), g4.x, acc[e][0]);
                    acc[e][1] = tgAddMin(tgLds1(xa + (ok ? co[1] : 0u)), g4.y, acc[e][1]);
                    acc[e][2] = tgAddMin(tgLds1(xa + (ok ? co[2] : 0u)), g4.z, acc[e][2]);
                    acc[e][3] = tgAddMin(tgLds1(xa + (ok ? co[3] : 0u)), g4.w, acc[e][3]);
                } else {
                    const uint32_t xv = tgLds1(xrow[e] + j4);   // x[k][j]: k sends to j
                    acc[e][0] = tgAddMin(xv, g4.x, acc[e][0]);
                    acc[e][1] = tgAddMin(xv, g4.y, acc[e][1]);
                    acc[e][2] = tgAddMin(xv, g4.z, acc[e][2]);
                    acc[e][3] = tgAddMin(xv, g4.w, acc[e][3]);
                }
            }
        }
#pragma unroll
        for (int e = 0; e < NSL; ++e) {
            const int s = s0 + e;
            if (s < nk) {
                // H row = [4 x INF | Wd values, H[b] at index b - lo4(R) | 8 x INF]
                const uint32_t hrow = i * uint32_t(nk) + uint32_t(s);
                const uint32_t hA = hAddr + hrow * HSB + 16u + ch * 16u;
                tgSts4(hA, make_uint4(acc[e][0], acc[e][1], acc[e][2], acc[e][3]));   // (the INF pads of the row: once per level, tgLevelBatched)
            }
        }
    }
}

// The island lists phase 2 works from, one thread per mask of the batch (the last threads of the CTA, during phase 1):
//   record of row (R, k) = { row-in-batch | lo4(S)/4 << 16 | (lo4(R) - lo4(S))/4 << 24 ,  S = R u {k} | k << 16 }
// filed at the next free position of island k's stretch (the stretches start at the prefix of the prepass counts).
// (Until round 2's last day the phase-1 item of chunk 0 filed its rows itself: those lanes sit in EVERY warp of the CTA --
// items are chunk-fastest --, so every warp paid the ~100 instructions and the shared-memory atomics of the filing on each pass.)
__device__ __forceinline__ void tgBuildLists(const TgShared& sm, const uint32_t* desc, uint2* list, int* cur, int nb, int nk) {
    const int Lw = sm.sWindowed ? sm.sL : 0;
    for (int i = TG_NT - 1 - int(threadIdx.x); i < nb; i += TG_NT) {
        const uint32_t* d = desc + i * TG_DESC_W;
        const uint32_t w0 = d[0], klLo = d[2], klHi = d[3];
        const uint32_t R = w0 & 0xffffu;
        const int cap = int(w0 >> 16);
        const int lo4R = max(0, Lw - cap) & ~3;
        for (int s = 0; s < nk; ++s) {
            const uint32_t k = tgNibble(klLo, klHi, s);
            const int lo4S = max(0, Lw - cap - int(sm.maxlenK[k])) & ~3;
            const int pos = atomicAdd(&cur[k], 1);
            list[pos] = make_uint2(uint32_t(i * nk + s) | uint32_t(lo4S >> 2) << 16 | uint32_t((lo4R - lo4S) >> 2) << 24, R | (1u << k) | k << 16);
        }
    }
}

// One block of 4 diagonals d = dq+1..dq+4 for one row and 4 starts a0..a0+3: LO = H[a0+dq .. a0+dq+3],
// HI = the next 4 values (loaded here); start a0+ai at diagonal d reads H[a0+ai+d].
#define TG_P2_STEP(LO, HI)                                                                     \
    {                                                                                          \
        const uint4 h = tgLds4(hA);                                                            \
        hA += 16;                                                                              \
        HI[0] = h.x; HI[1] = h.y; HI[2] = h.z; HI[3] = h.w;                                    \
        _Pragma("unroll") for (int e = 0; e < 4; ++e) {                                        \
            uint4 c4;                                                                          \
            if (GLOBALC) {                                                                     \
                const int d = dq + 1 + e;                                                      \
                c4 = make_uint4(TG_INFU, TG_INFU, TG_INFU, TG_INFU);                           \
                if (d <= dm && c < ((L - d + 3) >> 2)) {                                       \
                    c4 = TG_COST_AT4(I, sm.cdOff, cdkOff + tgGOff(L, d) + 4 * c, T);             \
                    const int amax = L - 1 - d;                                                \
                    c4.x = (a0 + 0 <= amax) ? c4.x : TG_INFU;                                  \
                    c4.y = (a0 + 1 <= amax) ? c4.y : TG_INFU;                                  \
                    c4.z = (a0 + 2 <= amax) ? c4.z : TG_INFU;                                  \
                    c4.w = (a0 + 3 <= amax) ? c4.w : TG_INFU;                                  \
                }                                                                              \
            } else {                                                                           \
                c4 = tgLds4(cA + e * cStride);                                                 \
            }                                                                                  \
            const uint32_t cv[4] = {c4.x, c4.y, c4.z, c4.w};                                   \
            _Pragma("unroll") for (int ai = 0; ai < 4; ++ai)                                   \
                out[ai] = tgAddMin(cv[ai], (ai + e + 1 < 4 ? LO[ai + e + 1] : HI[ai + e - 3]), out[ai]); \
        }                                                                                      \
        cA += 4 * cStride;                                                                     \
        dq += 4;                                                                               \
    }

// phase 2 of a batch.  Item = (row record e, chunk cw of 4 consecutive a), chunk fastest; the records are sorted by
// island (each island's stretch of the list was sized by the prepass).  Row (S, k) begins at start lo4S = lo4(cap(S));
// its H row begins at b = lo4R, so H[a + d] sits at stored index (a - lo4S) + d - delta, delta = lo4R - lo4S (a multiple of 4).
template <bool GLOBALC>
__device__ __forceinline__ void tgPhase2B(const TgSolveCtx& ctx, const TgShared& sm, const uint2* list, int nItems, uint32_t hAddr,
                                          uint32_t csBase, uint32_t* gBatch, int nbw, uint32_t mNbw, uint32_t HSB,
                                          uint32_t cStride, unsigned long long& bestKey) {
    const TgInstDev& I = ctx.inst[sm.sInst];
    const int L = sm.sL, Lp = sm.sLp, Wd = sm.sWd;
    const uint32_t T = sm.sT;
    for (int t = threadIdx.x; t < nItems; t += TG_NT) {
        const uint32_t e = tgDivM(uint32_t(t), mNbw);
        const int cw = int(uint32_t(t) - e * uint32_t(nbw));
        const uint2 info = list[e];
        const int k = int(info.y >> 16);
        const uint32_t hrow = info.x & 0xffffu;
        const int lo4S = int(info.x >> 16 & 0xffu) << 2, dq4 = int(info.x >> 24);
        const int a0 = lo4S + 4 * cw, c = a0 >> 2;   // c = absolute tile of 4 starts
        uint32_t out[4] = {TG_INFU, TG_INFU, TG_INFU, TG_INFU};
        if (a0 < Lp) {
            // blocks of 4 diagonals: from the first that reaches the H row to the last admissible one
            // (never past the end of the H row: such entries lie right of this row's window)
            const int dm = sm.dmaxTile[k][c], q0 = max(0, dq4 - 1 - cw);
            const int nq = min((dm + 3) >> 2, nbw - cw + dq4 + 1);
            if (q0 < nq) {
                const size_t cdkOff = size_t(sm.isl[k]) * I.triG;   // island k's table (L2 fallback of the cost rows)
                uint32_t hA = hAddr + hrow * HSB + 16u + uint32_t(4 * (cw + q0 - dq4)) * 4u;
                uint32_t cA = csBase + (sm.baseK[k] + uint32_t(a0)) * 4u + uint32_t(4 * q0) * cStride;
                int dq = 4 * q0;
                uint32_t Wa[4], Wb[4];
                {
                    const uint4 h = tgLds4(hA);
                    hA += 16;
                    Wa[0] = h.x; Wa[1] = h.y; Wa[2] = h.z; Wa[3] = h.w;
                }
#pragma unroll 1
                for (int q = q0; q < nq; q += 2) {
                    TG_P2_STEP(Wa, Wb)
                    if (q + 1 >= nq) break;
                    TG_P2_STEP(Wb, Wa)
                }
            }
        }
        *reinterpret_cast<uint4*>(gBatch + size_t(hrow) * Wd + 4 * cw) = make_uint4(out[0], out[1], out[2], out[3]);
        if (a0 == 0 && out[0] < TG_INFU) {
            const unsigned long long kk = (unsigned long long)out[0] << 32 | (unsigned long long)(info.y & 0xffffu) << 8 | (unsigned long long)k;
            bestKey = kk < bestKey ? kk : bestKey;
        }
    }
}

// One wavefront level for this CTA's share [lo, hi) of the level's masks (member `member` of a team of `teamSize`).
// Pipeline per batch n (two CTA barriers):
//   wait copies(n) | barrier | issue copies(n+1) ; phase 1(n) ; list cursors(n+1) | barrier | phase 2(n) ; prepass(n+2)
// Descriptors, source-row indices, island counts / cursors and source rows are double buffered; the list and the H rows
// are single.
__device__ void tgLevelBatched(const TgSolveCtx& ctx, TgShared& sm, uint32_t* dyn, const uint32_t* Gprev, uint32_t* Gcur,
                               unsigned long long* key, int Ke, int r, int member, int teamSize) {
    const int tid = threadIdx.x;
    const int Lp = sm.sLp, Wd = sm.sWd, nbw = Wd >> 2, nk = Ke - r;
    const int nMasks = sm.binom[Ke][r];
    const int lo = int((int64_t(nMasks) * member) / teamSize), hi = int((int64_t(nMasks) * (member + 1)) / teamSize);
    if (lo >= hi) return;
    const int HS = tgRowStride(Wd), SS = tgSrcStride(Wd);
    // split of the shared memory behind the cost rows for this level: computed by every thread (a few dozen instructions)
    // rather than by one thread and a CTA barrier; the island counts are zero on entry (cleared at the start of the item
    // and by cursors() for every batch that was counted)
    int NB, nsl, nsg;
    uint32_t oDesc[2], oSrcRow[2], oList, oH, oSrc[2];
    {
        const int avail = ctx.dynWords - sm.batchOff;
        const int perMask = nk * HS + 2 * r * SS + 2 * TG_DESC_W + 2 * r + 2 * nk;
        // (floor of the quotient through a float reciprocal rounded down, then corrected: no integer division)
        int fit = int(float(max(avail - 32, 0)) * __frcp_rd(float(perMask)));
        if ((fit + 1) * perMask <= avail - 32) ++fit;
        if (fit * perMask > avail - 32) --fit;
        NB = min(min(TG_NB_MAX, hi - lo), max(1, fit));
        // phase-1 items take NSL rows each: fewest CTA passes x instructions per item
        int best = 0, bestCost = 0x7fffffff;
#pragma unroll
        for (int lq = 0; lq <= 3; ++lq) {   // NSL = 1, 2, 4, 8 (TG_SPL)
            if ((1 << lq) > (sm.sNAct ? 4 : TG_SPL)) break;
            const int items = NB * nbw * ((nk + (1 << lq) - 1) >> lq);
            const int cost = ((items + TG_NT - 1) / TG_NT) * (3 + 5 * (1 << lq));
            if (cost < bestCost) { bestCost = cost; best = lq; }
        }
        nsl = 1 << best; nsg = (nk + nsl - 1) >> best;
        uint32_t o = uint32_t(sm.batchOff);
        for (int b = 0; b < 2; ++b) { oDesc[b] = o; o += uint32_t((NB * TG_DESC_W + 3) & ~3); }
        for (int b = 0; b < 2; ++b) { oSrcRow[b] = o; o += uint32_t((NB * r + 3) & ~3); }
        oList = o; o += uint32_t((2 * nk * NB + 3) & ~3);
        oH = o; o += uint32_t(NB * nk * HS);
        oSrc[0] = o; o += uint32_t(NB * r * SS);
        oSrc[1] = o;
    }
    const uint32_t mNbw = tgMagic(uint32_t(nbw)), mNsg = tgMagic(uint32_t(nsg));
    uint32_t* const descB[2] = {dyn + oDesc[0], dyn + oDesc[1]};
    uint32_t* const srcRowB[2] = {dyn + oSrcRow[0], dyn + oSrcRow[1]};
    uint2* const list = reinterpret_cast<uint2*>(dyn + oList);
    const uint32_t hAddr = tgSmemAddr(dyn + oH);
    const uint32_t srcAddr[2] = {tgSmemAddr(dyn + oSrc[0]), tgSmemAddr(dyn + oSrc[1])};
    const uint32_t HSB = uint32_t(HS) * 4u, SSB = uint32_t(SS) * 4u, cStride = uint32_t(Lp) * 4u;
    const bool actb = TG_VAR && sm.sNAct > 0;
    const uint32_t csBase = tgSmemAddr(dyn), xInfAddr = tgSmemAddr(&sm.xInf[0]);
    const uint32_t xsBase = actb ? tgSmemAddr(dyn + sm.xOff) : tgSmemAddr(&sm.xS[0][0]);
    const bool globalC = sm.useGlobalC != 0;
    const int nBatches = (hi - lo + NB - 1) / NB;
    unsigned long long bestKey = TG_KEY_NONE;
    // the prepass runs on the threads that get the fewest phase-2 items (the last ones)
    const int pi = TG_NT - 1 - tid;
    // list cursors of a batch = exclusive prefix of its island counts (lanes 0..15 of warp 0); the counts are cleared for
    // the prepass that reuses the buffer two batches later
    auto cursors = [&](int par) {
        if (tid < 32) {
            const int c = tid < Ke ? sm.cntP[par][tid] : 0;
            int inc = c;
#pragma unroll
            for (int o = 1; o < 16; o <<= 1) {
                const int a = __shfl_up_sync(0xffffffffu, inc, o);
                if ((tid & 15) >= o) inc += a;
            }
            if (tid < TG_MAX_K) { sm.cur[par][tid] = inc - c; sm.cntP[par][tid] = 0; }
        }
    };
    {   // H row = [4 x INF | Wd values, H[b] at index b - lo4(R) | 8 x INF]: the pads are the same for every batch of the level
        const uint4 inf4 = make_uint4(TG_INFU, TG_INFU, TG_INFU, TG_INFU);
        for (int w = tid; w < NB * nk; w += TG_NT) {
            const uint32_t rowA = hAddr + uint32_t(w) * HSB;
            tgSts4(rowA, inf4);
            tgSts4(rowA + 16u + uint32_t(nbw) * 16u, inf4);
            tgSts4(rowA + 32u + uint32_t(nbw) * 16u, inf4);
        }
    }
    for (int j = pi; j < 2 * NB; j += TG_NT) {   // the first two batches side by side: one mask a thread
        const int b = j >= NB ? 1 : 0, i = j - b * NB, m0 = lo + b * NB;
        if (i < hi - m0) tgPrepassMask(ctx, sm, descB[b] + i * TG_DESC_W, srcRowB[b] + i * r, sm.cntP[b], uint32_t(m0 + i), r, Ke);
    }
    __syncthreads();
    cursors(0);
    tgIssueBatch(srcRowB[0], srcAddr[0], Gprev, min(NB, hi - lo), r, Wd, nbw, mNbw, SSB);
    for (int n = 0; n < nBatches; ++n) {
        const int m0 = lo + n * NB, nb = min(NB, hi - m0), par = n & 1;
        asm volatile("cp.async.wait_all;" ::: "memory");
        __syncthreads();   // copies(n) have landed; descriptors / cursors of this batch are visible; phase 2 of batch n-1 is over
        if (n + 1 < nBatches) {
            tgIssueBatch(srcRowB[par ^ 1], srcAddr[par ^ 1], Gprev, min(NB, hi - m0 - NB), r, Wd, nbw, mNbw, SSB);
            cursors(par ^ 1);
        }
#define TG_P1_CASE(N, A) case N: tgPhase1B<N, A>(sm, descB[par], srcAddr[par], hAddr, nb, r, nk, nbw, nsg, mNbw, mNsg, SSB, HSB, xsBase, xInfAddr); break;
        if (actb) switch (nsl) { TG_P1_CASE(1, true) TG_P1_CASE(2, true) TG_P1_CASE(4, true) }   // (at most 4 rows an item with size classes)
        else switch (nsl) { TG_P1_CASE(1, false) TG_P1_CASE(2, false) TG_P1_CASE(4, false) TG_P1_CASE(8, false) }
#undef TG_P1_CASE
        tgBuildLists(sm, descB[par], list, sm.cur[par], nb, nk);
        __syncthreads();   // H rows and the island-sorted list of batch n are complete
        uint32_t* const gBatch = Gcur + size_t(m0) * nk * Wd;
        if (globalC) tgPhase2B<true>(ctx, sm, list, nb * nk * nbw, hAddr, csBase, gBatch, nbw, mNbw, HSB, cStride, bestKey);
        else tgPhase2B<false>(ctx, sm, list, nb * nk * nbw, hAddr, csBase, gBatch, nbw, mNbw, HSB, cStride, bestKey);
        if (n + 2 < nBatches) {
            const int m2 = m0 + 2 * NB;
            for (int i = pi; i < min(NB, hi - m2); i += TG_NT)
                tgPrepassMask(ctx, sm, descB[par] + i * TG_DESC_W, srcRowB[par] + i * r, sm.cntP[par], uint32_t(m2 + i), r, Ke);
        }
    }
    if (__any_sync(0xffffffffu, bestKey != TG_KEY_NONE)) {
        for (int o = 16; o > 0; o >>= 1) {
            const unsigned long long ot = __shfl_xor_sync(0xffffffffu, bestKey, o);
            bestKey = ot < bestKey ? ot : bestKey;
        }
        if ((tid & 31) == 0) atomicMin(key, bestKey);
    }
}

// ---------------------------------------------------------------------------------------------
// Levels r >= 1 of a DP that a TEAM of CTAs shares (few instances: cfg3 / cfg4): one WARP (or half warp) per mask, streaming
// over its strided share of the level's masks (colexicographic rank order); nothing but the item's staged tables is
// shared between the warps of a CTA, so a level needs no CTA barrier at all.  Per mask R (|R| = r, nk = Ke - r):
//   issue   16-byte cp.async copies of the r source rows G_{r-1}[R\{j}][j][.] into the warp's
//           shared-memory buffer, one mask ahead of their use (double buffer, commit / wait_group)
//   phase 1 H[R][k][b] = min_{j in R} x[k][j] + src[j][b]       lane = (4 consecutive b) x (k group)
//   phase 2 G_r[R][k][a] = min_{b>a} Cs_k[a][b] + H[R][k][b]    lane = (4 consecutive a) x (k group)
// A team's share of a level is dozens of small batches per CTA; measured at cfg4 the CTA-wide batches above (1.60 ms),
// the same batches per warp (2.04 ms) and this streaming form (1.40 ms), so the team keeps it.
// ---------------------------------------------------------------------------------------------
// phase 1 for the NSL k slots  slot0, slot0+NG, ...  of this lane's island group and its b chunks:
//   H[R][k][b] = min_{j in R} x[k][j] + src[j][b],  written to the warp's H rows.
// All slots but the last are valid for every lane; an invalid last slot reads an all-INF x row.
template <int NSL, bool ACTB>
__device__ __forceinline__ void tgPhase1W(const TgShared& sm, uint32_t R, int r, int nk, int nb4, int c0, int CH, int NG,
                                         int slot0, uint32_t srcAddr, uint32_t rowBytes, uint32_t hAddr0, const uint8_t* kl,
                                         uint32_t xsBase, uint32_t xInfAddr, int lo4R) {
    uint32_t xrow[NSL];
#pragma unroll
    for (int i = 0; i < NSL; ++i) {
        const int s = slot0 + NG * i;
        xrow[i] = (i + 1 < NSL || s < nk) ? xsBase + uint32_t(kl[s]) * (TG_MAX_K * 4u) : xInfAddr;
    }
    const bool lastValid = slot0 + NG * (NSL - 1) < nk;
    for (int c = c0; c < nb4; c += CH) {
        uint32_t acc[NSL][4];
#pragma unroll
        for (int i = 0; i < NSL; ++i) { acc[i][0] = acc[i][1] = acc[i][2] = acc[i][3] = TG_INFU; }
        uint32_t co[4] = {0, 0, 0, 0};
        if (ACTB) {
#pragma unroll
            for (int cq = 0; cq < 4; ++cq) co[cq] = uint32_t(sm.clsOfS[min(lo4R + 4 * c + cq, 255)]) * (TG_MAX_K * TG_MAX_K * 4u);
        }
        uint32_t sA = srcAddr + uint32_t(c) * 16u;
        uint32_t Rb = R;
#pragma unroll 2
        for (int ji = 0; ji < r; ++ji) {
            const uint32_t j4 = uint32_t(__ffs(Rb) - 1) * 4u;
            Rb &= Rb - 1;
            const uint4 g4 = tgLds4(sA);
            sA += rowBytes;
#pragma unroll
            for (int i = 0; i < NSL; ++i) {
                if (ACTB) {   // per-boundary activation sizes: the transfer matrix of each of the chunk's 4 boundaries
                    const bool ok = i + 1 < NSL || lastValid;
                    const uint32_t xa = xrow[i] + j4;
                    acc[i][0] = tgAddMin(tgLds1(xa + (ok ? co[0] : 0u)), g4.x, acc[i][0]);
                    acc[i][1] = tgAddMin(tgLds1(xa + (ok ? co[1] : 0u)), g4.y, acc[i][1]);
                    acc[i][2] = tgAddMin(tgLds1(xa + (ok ? co[2] : 0u)), g4.z, acc[i][2]);
                    acc[i][3] = tgAddMin(tgLds1(xa + (ok ? co[3] : 0u)), g4.w, acc[i][3]);
                } else {
                    const uint32_t xv = tgLds1(xrow[i] + j4);   // x[k][j]: k sends to j
                    acc[i][0] = tgAddMin(xv, g4.x, acc[i][0]);
                    acc[i][1] = tgAddMin(xv, g4.y, acc[i][1]);
                    acc[i][2] = tgAddMin(xv, g4.z, acc[i][2]);
                    acc[i][3] = tgAddMin(xv, g4.w, acc[i][3]);
                }
            }
        }
#pragma unroll
        for (int i = 0; i < NSL; ++i) {
            if (i + 1 < NSL || lastValid) {
                // H row = [4 x INF | Wd values, H[b] at index b - lo4R | 8 x INF]
                const uint32_t hA = hAddr0 + uint32_t(slot0 + NG * i) * rowBytes + 16u + uint32_t(c) * 16u;
                tgSts4(hA, make_uint4(acc[i][0], acc[i][1], acc[i][2], acc[i][3]));   // (the INF pads: once per level, tgWarpLevel)
            }
        }
    }
}

// phase 2 for this lane's rows (slots g, g+NG, ...) and a chunks of mask R:
//   G_r[R][k][a] = min_{b>a} Cs_k[a][b] + H[R][k][b]
// Row of (R u {k}, k) starts at start lo4S = lo4(capR + maxlen_k); the H row starts at b = lo4R, so
// H[a + d] sits at stored index (a - lo4S) + d - delta, delta = lo4R - lo4S (a multiple of 4).
template <bool GLOBALC>
__device__ __forceinline__ void tgPhase2W(const TgSolveCtx& ctx, const TgShared& sm, uint32_t R, int capR, int nk, int nbw, int c0,
                                         int CH, int NG, int g, uint32_t hAddr0, uint32_t rowBytes, uint32_t csBase,
                                         uint32_t cStride, const uint8_t* kl, uint32_t* gRow, unsigned long long& bestKey) {
    const TgInstDev& I = ctx.inst[sm.sInst];
    const int L = sm.sL, Lp = sm.sLp, Wd = sm.sWd;
    const uint32_t T = sm.sT;
    const int Lw = sm.sWindowed ? L : 0;              // lo4(cap) = floor4(max(0, Lw - cap)): 0 when rows are not windowed
    const int lo4R = max(0, Lw - capR) & ~3;
    for (int s = g; s < nk; s += NG) {
        const int k = kl[s];
        const int lo4S = max(0, Lw - capR - int(sm.maxlenK[k])) & ~3, dq4 = (lo4R - lo4S) >> 2;
        const size_t cdkOff = size_t(sm.isl[k]) * I.triG;   // island k's table (L2 fallback of the cost rows)
        const uint32_t cBase = csBase + (sm.baseK[k] + uint32_t(lo4S)) * 4u, hRow = hAddr0 + uint32_t(s) * rowBytes + 16u;
        uint32_t* const gOut = gRow + size_t(s) * Wd;
        for (int cw = c0; cw < nbw; cw += CH) {
            const int a0 = lo4S + 4 * cw, c = a0 >> 2;   // c = absolute tile of 4 starts
            uint32_t out[4] = {TG_INFU, TG_INFU, TG_INFU, TG_INFU};
            if (a0 < Lp) {
                // blocks of 4 diagonals: from the first that reaches the H row to the last admissible one
                // (never past the end of the H row: such entries lie right of this row's window)
                const int dm = sm.dmaxTile[k][c], q0 = max(0, dq4 - 1 - cw);
                const int nq = min((dm + 3) >> 2, nbw - cw + dq4 + 1);
                if (q0 < nq) {
                    uint32_t hA = hRow + uint32_t(4 * (cw + q0 - dq4)) * 4u;
                    uint32_t cA = cBase + uint32_t(cw) * 16u + uint32_t(4 * q0) * cStride;
                    int dq = 4 * q0;
                    uint32_t Wa[4], Wb[4];
                    {
                        const uint4 h = tgLds4(hA);
                        hA += 16;
                        Wa[0] = h.x; Wa[1] = h.y; Wa[2] = h.z; Wa[3] = h.w;
                    }
#pragma unroll 1
                    for (int q = q0; q < nq; q += 2) {
                        TG_P2_STEP(Wa, Wb)
                        if (q + 1 >= nq) break;
                        TG_P2_STEP(Wb, Wa)
                    }
                }
            }
            *reinterpret_cast<uint4*>(gOut + 4 * cw) = make_uint4(out[0], out[1], out[2], out[3]);
            if (a0 == 0 && out[0] < TG_INFU) {
                const unsigned long long kk = (unsigned long long)out[0] << 32 | (unsigned long long)(R | (1u << k)) << 8 | (unsigned long long)k;
                bestKey = kk < bestKey ? kk : bestKey;
            }
        }
    }
}

// One wavefront level for this warp's share of the masks.  SW = 32: one mask at a time on the whole warp.
// SW = 16: two masks side by side, one per half warp (narrow row windows leave most of a full warp idle and
// the per-mask bookkeeping -- copies, windows, complement list -- then costs more than the relaxations;
// two masks share every one of those instructions).  Each sub-warp has its own H rows and source buffers
// inside the warp's buffer.
// The masks are dealt out STRIDED and looked up in the rank tables: sub-warp q of Q takes the masks of rank
// q, q+Q, q+2Q, ...  (Rounds 1 and 2 gave every warp a contiguous run of ranks, walked with Gosper's successor, the source
// ranks from two 16-lane scans of binomials: 13.6 % of the kernel's instructions at cfg4.)
// That arithmetic is replaced by the device tables (maskOf: rank -> mask, rankOf: mask -> rank), read three and two masks
// ahead of their use so that their L2 latency is covered by the masks in between: iteration `it` computes mask it, issues
// the copies of mask it+1, loads the source ranks of mask it+2 and the mask it+3.  A strided share also samples the level
// evenly (a run of colexicographic ranks shares its high islands, whose admissible diagonals differ by up to 19:1).
// Measured at cfg4: solver 1.393 -> 1.342 ms, the levels' share of the CTA cycles 69 -> 66 %.
// The first trips of a (sub-)warp in a level: masks of trips 0..2 and the source ranks of trips 0..1 (sw = lanes per mask of
// that level, 16 or 32).  Looked up BEFORE the wait for the previous level's team barrier: the two dependent table
// look-ups (mask, then ranks) overlap the wait instead of following it.
struct TgPre { uint32_t R0, R1, R2, rk0, rk1; };
__device__ __forceinline__ TgPre tgPreLookup(const TgSolveCtx& ctx, const TgShared& sm, int Ke, int r, int gw, int GW, int sw) {
    const int lane = threadIdx.x & 31;
    const int M = 32 / sw, sub = sw == 32 ? 0 : (lane >> 4), sl = lane & (sw - 1);
    const int nMasks = sm.binom[Ke][r];
    const int q = gw * M + sub, Q = GW * M;
    const uint16_t* mtab = ctx.maskOf + tgPopOff[r];
    const uint32_t myBit = sl < TG_MAX_K ? (1u << sl) : 0u;
    TgPre P;
    P.R0 = q < nMasks ? uint32_t(__ldg(mtab + q)) : 0u;
    P.R1 = q + Q < nMasks ? uint32_t(__ldg(mtab + q + Q)) : 0u;
    P.R2 = q + 2 * Q < nMasks ? uint32_t(__ldg(mtab + q + 2 * Q)) : 0u;
    P.rk0 = (P.R0 & myBit) ? uint32_t(__ldg(ctx.rankOf + (P.R0 ^ myBit))) : 0u;   // lane sl in R: rank of R \ {sl}
    P.rk1 = (P.R1 & myBit) ? uint32_t(__ldg(ctx.rankOf + (P.R1 ^ myBit))) : 0u;
    return P;
}

template <int SW>
__device__ __forceinline__ void tgIssueMaskT(uint32_t R, uint32_t rk, bool valid, int r, int nk, int Wd, int nbw, int cpShift,
                                             uint32_t bufAddr, uint32_t rowBytes, const uint32_t* Gprev, uint32_t* rowOf, int lane) {
    const int sl = lane & (SW - 1);
    const bool member = valid && sl < TG_MAX_K && ((R >> sl) & 1u);
    const int p = __popc(R & ((1u << sl) - 1u));
    if (member) rowOf[p] = rk * uint32_t(nk + 1) + uint32_t(sl - p);   // row of state (R\{sl}, first island sl) in level r-1
    __syncwarp();
    if (valid) {
        const int CP = 1 << cpShift;   // chunks per row, rounded up to a power of two
        for (int w = sl; w < (r << cpShift); w += SW) {
            const int ji = w >> cpShift, ch = w & (CP - 1);
            if (ch < nbw) {
                const uint32_t* src = Gprev + size_t(rowOf[ji]) * Wd + 4 * ch;
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(bufAddr + uint32_t(ji) * rowBytes + uint32_t(ch) * 16u), "l"(src) : "memory");
            }
        }
    }
}

template <int SW>
__device__ void tgWarpLevel(const TgSolveCtx& ctx, TgShared& sm, const uint32_t* Cs, uint32_t* wbuf, const uint32_t* Gprev,
                            uint32_t* Gcur, unsigned long long* key, int Ke, int r, int gw, int GW, const TgPre pre) {
    constexpr int M = 32 / SW, SWSH = SW == 32 ? 5 : 4;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int sub = lane >> SWSH, sl = lane & (SW - 1);
    const int Lp = sm.sLp, Wd = sm.sWd, nbw = Wd >> 2, nk = Ke - r;
    const int HS = tgRowStride(Wd);
    const int nMasks = sm.binom[Ke][r];
    const int q = gw * M + sub, Q = GW * M;
    if (gw * M >= nMasks) return;                                        // (sub-warp 0 of a warp has the most masks)
    const int per = (nMasks - 1 - gw * M) / Q + 1;                       // masks of sub-warp 0 = trips of the warp
    const int cnt = q < nMasks ? (nMasks - 1 - q) / Q + 1 : 0;           // masks of this sub-warp (per or per - 1)
    // sub-lane = (chunk of 4 starts) x (island group): CH chunk lanes, NG = SW / CH groups
    const int cpShift = nbw <= 2 ? 1 : (nbw <= 4 ? 2 : (nbw <= 8 ? 3 : (nbw <= 16 ? 4 : (nbw <= 32 ? 5 : 6))));
    const int chShift = min(cpShift, SWSH);
    const int CH = 1 << chShift, NG = SW >> chShift;
    const int c0 = sl & (CH - 1), g = sl >> chShift;
    const uint32_t rowBytes = uint32_t(HS) * 4u, cStride = uint32_t(Lp) * 4u;
    const uint32_t hAddr0 = tgSmemAddr(wbuf) + uint32_t(sub) * uint32_t(nk + 2 * r) * rowBytes;
    const bool actb = TG_VAR && sm.sNAct > 0;
    const uint32_t csBase = tgSmemAddr(Cs), xsBase = actb ? tgSmemAddr(Cs + sm.xOff) : tgSmemAddr(&sm.xS[0][0]);
    const uint32_t xInfAddr = tgSmemAddr(&sm.xInf[0]);
    const uint32_t bufAddr[2] = {hAddr0 + uint32_t(nk) * rowBytes, hAddr0 + uint32_t(nk + r) * rowBytes};
    uint32_t* rowOf = &sm.rowOf[warp][sub * TG_MAX_K];
    uint8_t* kl = &sm.kl[warp][sub * TG_MAX_K];
    const uint32_t keMask = (1u << Ke) - 1u;
    const bool globalC = sm.useGlobalC != 0;
    unsigned long long bestKey = TG_KEY_NONE;

    {   // the INF pads of the sub-warp's H rows (4 words before, 8 behind the Wd values): the same for every mask of the level
        const uint4 inf4 = make_uint4(TG_INFU, TG_INFU, TG_INFU, TG_INFU);
        for (int s = sl; s < nk; s += SW) {
            const uint32_t rowA = hAddr0 + uint32_t(s) * rowBytes;
            tgSts4(rowA, inf4);
            tgSts4(rowA + 16u + uint32_t(nbw) * 16u, inf4);
            tgSts4(rowA + 32u + uint32_t(nbw) * 16u, inf4);
        }
        __syncwarp();
    }
    const uint16_t* mtab = ctx.maskOf + tgPopOff[r];
    const uint32_t myBit = sl < TG_MAX_K ? (1u << sl) : 0u;
    uint32_t R = pre.R0, R1 = pre.R1, R2 = pre.R2;   // masks of trips 0..2 (0 = none), looked up by the caller (tgPreLookup)
    uint32_t rk = pre.rk0, rk1 = pre.rk1;            // lane sl in R: rank of R \ {sl}
    tgIssueMaskT<SW>(R, rk, cnt > 0, r, nk, Wd, nbw, cpShift, bufAddr[0], rowBytes, Gprev, rowOf, lane);
    asm volatile("cp.async.commit_group;" ::: "memory");
    int b = 0;
    for (int it = 0; it < per; ++it, b ^= 1) {
        const int idx = q + it * Q;
        const bool valid = it < cnt, more = it + 1 < cnt;
        tgIssueMaskT<SW>(R1, rk1, more, r, nk, Wd, nbw, cpShift, bufAddr[b ^ 1], rowBytes, Gprev, rowOf, lane);
        asm volatile("cp.async.commit_group;" ::: "memory");   // possibly empty: keeps the group count uniform
        const uint32_t rk2 = (it + 2 < cnt && (R2 & myBit)) ? uint32_t(__ldg(ctx.rankOf + (R2 ^ myBit))) : 0u;
        const uint32_t R3 = it + 3 < cnt ? uint32_t(__ldg(mtab + idx + 3 * Q)) : 0u;
        const uint32_t comp = ~R & keMask;
        if (valid && sl < Ke && (comp >> sl & 1u)) kl[__popc(comp & ((1u << sl) - 1u))] = uint8_t(sl);
        const int capR = int(sm.capLo[R & 255u]) + int(sm.capHi[R >> 8]);   // cap(R) = sum of the members' longest slices
        asm volatile("cp.async.wait_group 1;" ::: "memory");   // this mask's rows have landed (the next mask's may be in flight)
        __syncwarp();

        // ---- phase 1: transfer pre-minimum, H rows into the sub-warp's shared memory -----------
        if (valid) {
            const int spl = actb ? 4 : TG_SPL;   // (the per-boundary variant keeps 4 transfer offsets more per lane)
            for (int s0 = 0; s0 < nk; s0 += NG * spl) {
                const int nsl = min(spl, (nk - s0 + NG - 1) >> (SWSH - chShift));   // slots of the widest island group
#define TG_P1_CASE(N, A) case N: tgPhase1W<N, A>(sm, R, r, nk, nbw, c0, CH, NG, s0 + g, bufAddr[b], rowBytes, hAddr0, kl, xsBase, xInfAddr, lo4Rw); break;
                const int lo4Rw = tgLo4(sm, capR);
                if (actb) switch (nsl) { TG_P1_CASE(1, true) TG_P1_CASE(2, true) TG_P1_CASE(3, true) TG_P1_CASE(4, true) }
                else switch (nsl) {
                    TG_P1_CASE(1, false) TG_P1_CASE(2, false) TG_P1_CASE(3, false) TG_P1_CASE(4, false)
                    TG_P1_CASE(5, false) TG_P1_CASE(6, false) TG_P1_CASE(7, false) TG_P1_CASE(8, false)
                }
#undef TG_P1_CASE
            }
        }
        __syncwarp();

        // ---- phase 2: min-plus product with the thresholded cost rows ----------------------------
        if (valid) {
            uint32_t* const gRow = Gcur + size_t(idx) * nk * Wd;
            if (globalC) tgPhase2W<true>(ctx, sm, R, capR, nk, nbw, c0, CH, NG, g, hAddr0, rowBytes, csBase, cStride, kl, gRow, bestKey);
            else tgPhase2W<false>(ctx, sm, R, capR, nk, nbw, c0, CH, NG, g, hAddr0, rowBytes, csBase, cStride, kl, gRow, bestKey);
        }
        __syncwarp();
        R = R1; R1 = R2; R2 = R3; rk1 = rk2;
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    if (__any_sync(0xffffffffu, bestKey != TG_KEY_NONE)) {
        for (int o = 16; o > 0; o >>= 1) {
            const unsigned long long ot = __shfl_xor_sync(0xffffffffu, bestKey, o);
            bestKey = ot < bestKey ? ot : bestKey;
        }
        if (lane == 0) atomicMin(key, bestKey);
    }
}

// ---------------------------------------------------------------------------------------------
// Step 7: plan back-tracker.  One warp, right after a DP that kept every level: re-derive the
// per-state argmin (lowest b, then lowest j — SURVEY A13) along the optimal path from the stored
// G levels of the slot.
// ---------------------------------------------------------------------------------------------
__device__ void tgBacktrack(const TgSolveCtx& ctx, const TgShared& sm, const TgItem* itp, unsigned long long key, const uint32_t* slot,
                            tg_result* out) {
    const int lane = threadIdx.x & 31;
    TgInstDev& I = ctx.inst[__ldcg(&itp->inst)];
    const int L = I.L, K = I.K, Ke = sm.sKe;
    const uint32_t T = __ldcg(&itp->T);
    uint8_t isl[TG_MAX_K];
#pragma unroll
    for (int e = 0; e < TG_MAX_K; ++e) isl[e] = sm.isl[e];
    const int64_t Trep = (T == TG_TINF) ? int64_t(TG_INF) : int64_t(T);
    if (key == TG_KEY_NONE) {
        if (lane == 0) {
            tg_result z;
            memset(&z, 0, sizeof(z));
            z.iter_time_us = INT64_MAX;
            z.n_thresholds_run = uint32_t(I.nrun + 1);
            *out = z;
        }
        return;
    }
    const uint32_t val = uint32_t(key >> 32);
    uint32_t S = uint32_t(key >> 8) & 0xffffu;
    int k = int(key & 0xffu);
    uint32_t R = S ^ (1u << k);
    int a = 0, n = 0;
    int sb[TG_MAX_K], si[TG_MAX_K], sp[TG_MAX_K];
    bool bad = false;
    while (true) {
        const int ko = isl[k];
        int b;
        if (R == 0) {
            b = L;
        } else {
            const int r = __popc(R);
            const int Wd = sm.sWd;
            const uint32_t* Gl = slot + tgLevelOff(0, Ke, Wd, r - 1);
            // this stage is followed by r later ones: its cost and plan come from the table of depth r + 1
            const size_t dq = (TG_VAR && I.nDepth > 1) ? size_t(r) : 0;
            int capR = 0;   // every source row (R\{j}, j) starts at start lo4(cap(R))
            for (int j = 0; j < Ke; ++j) if (R >> j & 1u) capR += sm.maxlenK[j];
            const int lo4R = tgLo4(sm, capR);
            unsigned long long best = TG_KEY_NONE;
            int bestLayer = 0;   // NEXT-2: the cost step the winning slice took (selects its plan)
            // lanes over (member j, boundary b) pairs, b inside the source rows' window: every load is independent
            const int bLo = max(a + 1, lo4R), nb = min(L - 1, lo4R + Wd - 1) - bLo + 1;
            for (int p = lane; p < nb * r; p += 32) {
                const int ji = p / nb, bb = bLo + (p - ji * nb);
                int layer = 0;
                const uint32_t c = TG_COST_AT(I, dq * K * I.triG, size_t(ko) * I.triG + tgGOff(L, bb - a) + a, T, &layer);
                if (c >= TG_INFU) continue;
                const int j = int(__fns(R, 0, ji + 1));
                const uint32_t Rp = R ^ (1u << j);
                const size_t row = size_t(ctx.rankOf[Rp]) * (Ke - r + 1) + (j - __popc(R & ((1u << j) - 1u)));
                const uint32_t xv = (TG_VAR && I.nAct) ? I.xAct[int(I.clsOf[bb]) * (TG_MAX_K * TG_MAX_K) + ko * TG_MAX_K + isl[j]] : I.x[ko * TG_MAX_K + isl[j]];
                if (I.xbound && xv > T) continue;
                const uint32_t v = c + xv + __ldcg(Gl + row * Wd + (bb - lo4R));
                if (v >= TG_INFU) continue;
                // lowest value, then lowest b, then lowest j
                const unsigned long long kk = (unsigned long long)v << 32 | (unsigned long long)bb << 8 | (unsigned long long)j;
                if (kk < best) { best = kk; bestLayer = layer; }
            }
            for (int o = 16; o > 0; o >>= 1) {
                const unsigned long long ot = __shfl_xor_sync(0xffffffffu, best, o);
                const int ol = __shfl_xor_sync(0xffffffffu, bestLayer, o);
                if (ot < best) { best = ot; bestLayer = ol; }
            }
            if (best == TG_KEY_NONE) { bad = true; break; }
            b = int(best >> 8) & 0xffffff;
            const int j = int(best & 0xffu);
            const size_t tbl = (TG_VAR && I.nLayers) ? size_t(bestLayer) : dq;   // (the layer depends on (a, b, k) only: every lane with the winning b agrees)
            sb[n] = a; si[n] = ko; sp[n] = I.argp[tbl * size_t(I.NS) * K + size_t(tgSliceIdx(L, a, b)) * K + ko];
            ++n;
            a = b; k = j; R ^= 1u << j;
            continue;
        }
        int lastLayer = 0;
        TG_COST_AT(I, 0, size_t(ko) * I.triG + tgGOff(L, b - a) + a, T, &lastLayer);
        sb[n] = a; si[n] = ko; sp[n] = I.argp[size_t(lastLayer) * I.NS * K + size_t(tgSliceIdx(L, a, b)) * K + ko];
        ++n;
        break;
    }
    if (bad) atomicExch(&ctx.ctrl->errFlag, 2);
    if (lane == 0) {
        tg_result z;
        memset(&z, 0, sizeof(z));
        uint32_t So = 0;
        for (int e = 0; e < Ke; ++e) if (S >> e & 1u) So |= 1u << isl[e];
        z.sum_us = val;
        z.island_mask = So;
        z.n_stages = n;
        z.n_thresholds_run = uint32_t(I.nrun + 1);
        z.bottleneck_us = int32_t(Trep);
        z.iter_time_us = int64_t(val) + int64_t(I.m - 1) * Trep;   // (= the incumbent's value when this is the final DP)
        for (int e = 0; e < n; ++e) { z.stage_begin[e] = sb[e]; z.stage_island[e] = si[e]; z.stage_plan[e] = sp[e]; }
        *out = z;
    }
}

// ---------------------------------------------------------------------------------------------
// One DP(T): all wavefront levels of one item by a team of `teamSize` CTAs (this CTA = `member`).
// ---------------------------------------------------------------------------------------------
__device__ void tgRunItem(const TgSolveCtx& ctx, TgShared& sm, uint32_t* Cs, uint32_t* wbufAll, const TgItem* itp,
                          unsigned long long* key, int member, int teamSize, int slotIdx, int itemIdx) {
    tgStageItem(ctx, sm, Cs, wbufAll, itp, member == 0, teamSize > 1);
    tgMark(sm, 0);
    const TgInstDev& I = ctx.inst[sm.sInst];
    const int Ke = sm.sSlack >= 0 ? sm.sKe : 0;   // the islands' longest slices cannot cover L layers: infeasible at T
    const int Wd = sm.sWd;
    uint64_t bufWords = 0;   // words of one ping-pong half; 0 = keep every level (a back-track follows)
    if (Ke > 0 && !(__ldcg(&itp->flags) & 1)) {
        uint32_t mx = 1;
        for (int q = 0; q < Ke; ++q) mx = max(mx, tgLevelRows(Ke, q));
        bufWords = uint64_t(mx) * uint64_t(sm.sLp);
    }
    uint32_t* slot = ctx.scratch + uint64_t(slotIdx) * ctx.slotWords;
    uint32_t* bar = ctx.slotBar + slotIdx;
    uint32_t arrivals = 0;
    bool pendingBar = false;
    if (Ke > 0) {
        if (threadIdx.x < 2 * TG_MAX_K) (&sm.cntP[0][0])[threadIdx.x] = 0;   // island counts of the batched levels: zero at every level's entry
        tgLevel0(ctx, sm, slot, key, member == 0);
        __syncthreads();
        for (int r = 1; r < Ke; ++r) {
            const uint32_t* Gprev = slot + tgLevelOff(bufWords, Ke, Wd, r - 1);
            uint32_t* Gcur = slot + tgLevelOff(bufWords, Ke, Wd, r);
            if (TG_VAR && I.nDepth > 1) tgStageCosts(ctx, sm, Cs, r + 1, false);   // stages of this level hold r + 1 microbatches
            if (teamSize > 1) {
                const int warp = threadIdx.x >> 5, nW = sm.nWarps;
                TgPre pre = {0u, 0u, 0u, 0u, 0u};
                const bool pairL = (Wd >> 2) <= 16 && 2 * (Ke + r) * tgRowStride(Wd) <= sm.wbufWords && int(sm.binom[Ke][r]) > teamSize * nW;
                if (warp < nW) pre = tgPreLookup(ctx, sm, Ke, r, member * nW + warp, teamSize * nW, pairL ? 16 : 32);
                if (pendingBar) { tgTeamWait(bar, arrivals); pendingBar = false; tgMark(sm, 4); }   // level r-1 is complete on every member
                if (warp < nW) {
                    uint32_t* wbuf = wbufAll + sm.wbufOff + size_t(warp) * sm.wbufWords;
                    // two masks per warp when the windows are narrow and both masks' rows fit the warp's buffer
                    // ... and the level has more masks than the team has warps (else a mask gets the whole warp: the small
                    // levels at both ends of a DP are one trip of pure latency -- cfg3 0.506 -> 0.478 ms, cfg4 1.343 -> 1.327 ms)
                    const bool pair = (Wd >> 2) <= 16 && 2 * (Ke + r) * tgRowStride(Wd) <= sm.wbufWords && int(sm.binom[Ke][r]) > teamSize * nW;
                    if (pair) tgWarpLevel<16>(ctx, sm, Cs, wbuf, Gprev, Gcur, key, Ke, r, member * nW + warp, teamSize * nW, pre);
                    else tgWarpLevel<32>(ctx, sm, Cs, wbuf, Gprev, Gcur, key, Ke, r, member * nW + warp, teamSize * nW, pre);
                }
            } else {
                tgLevelBatched(ctx, sm, wbufAll, Gprev, Gcur, key, Ke, r, member, teamSize);
            }
            tgMark(sm, 3);
            // (after the last level of a DP that is not back-tracked nothing reads the team's rows: the round's grid barrier
            // is the next thing every member does, so the team barrier is left out)
            // Between two levels the barrier is split: arrive here, wait at the start of the next level behind its look-ups.
            if (teamSize > 1 && r + 1 < Ke) { arrivals += uint32_t(teamSize); tgTeamArrive(bar); pendingBar = true; }
            else if (teamSize > 1 && bufWords == 0) { arrivals += uint32_t(teamSize); tgTeamBarrier(bar, arrivals); }
            else __syncthreads();
            tgMark(sm, 4);
        }
    }
    tgMark(sm, 0);
    if ((__ldcg(&itp->flags) & TG_IT_TRACK) && member == 0 && threadIdx.x < 32)
        tgBacktrack(ctx, sm, itp, __ldcg(key), slot,
                    (__ldcg(&itp->flags) & TG_IT_SPEC) ? ctx.specOut + itemIdx : ctx.out + __ldcg(&itp->inst));
    __syncthreads();
    tgMark(sm, 7);
}

// DPs per round an instance with K islands should run: enough that every warp of a team (grid / DPs)
// has about eight masks at the widest level, but few enough that little of a round is speculation:
// measured best at 8 (cfg4, K = 16) to 10-12 (cfg3, K = 12) probes a round.
__device__ __forceinline__ int tgWish(const TgSolveCtx& ctx, int K) {
    const int widest = tgBinom[K][K >> 1];
    const int team = max(1, widest / (8 * TG_NW));
    return min(max(int(gridDim.x) / team, ctx.wishFloor), ctx.wishCap);
}

// ---------------------------------------------------------------------------------------------
// Scheduler (CTA 0): fold results of the previous round, plan the next one.  Exact search over the
// candidate thresholds cand[0..n) (reading R-search); f_T = best sum at T is
// non-increasing in T and feasibility is monotone in T:
//   FEAS   find the lowest feasible candidate: galloping from the necessary-condition index
//          lbIdx, then multi-section inside the bracket (loInf, hiFeas]
//   BNB    branch and bound over the remaining candidates: for c between two evaluated points
//          i < c < j,  iter_c >= f_j + (m-1) T_c  (f_c >= f_j); above the last evaluated point
//          iter_c >= (m-1) T_c.  A candidate is dropped when its bound cannot beat the incumbent
//          = lexicographic min of (iter, candidate index) over every DP evaluated, which is what
//          the full ascending sweep with strict improvement returns (lowest T wins ties).
//          Unresolved stretches are probed at evenly spaced points that include their right end.
//   SWEEP  (TG_SOLVE_FULL_SWEEP) every candidate in ascending order
//   FINAL  DP at T* keeping every level, followed by the back-track
// ---------------------------------------------------------------------------------------------
// could candidate c, whose sum is at least lbF, still beat the incumbent?
// (the incumbent and the candidate list, read once into registers: the scheduler is a single thread per
// instance and every field of TgInstDev it touches is a memory access)
// CTA-wide copy of n words of read-only global memory into shared memory, eight loads of a thread in flight (a plain
// `dst[w] = src[w]` loop through generic pointers is compiled as load, store, load, ...: one L2 round trip per word)
__device__ __forceinline__ void tgCopyToShared(uint32_t* dst, const uint32_t* src, int n) {
    for (int w0 = threadIdx.x; w0 < n; w0 += 8 * TG_NT) {
        uint32_t v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) v[u] = w0 + u * TG_NT < n ? __ldg(src + w0 + u * TG_NT) : 0u;
#pragma unroll
        for (int u = 0; u < 8; ++u) if (w0 + u * TG_NT < n) dst[w0 + u * TG_NT] = v[u];
    }
}

struct TgInc {
    int64_t incIter, m1;
    int incIdx;
    const uint32_t* cand;
    const uint32_t* win;   // cand[winLo .. winLo + winN) in shared memory (or null)
    int winLo, winN;
};
__device__ __forceinline__ bool tgBeats(const TgInc& B, int64_t lbF, int c) {
    if (B.incIdx < 0) return true;
    const unsigned off = unsigned(c - B.winLo);
    const uint32_t Tc = off < unsigned(B.winN) ? B.win[off] : __ldg(B.cand + c);   // cand is read-only during the solve
    const int64_t lb = lbF + B.m1 * int64_t(Tc);
    return lb < B.incIter || (lb == B.incIter && c < B.incIdx);
}

// last c in [lo, hi] with tgBeats(lbF, c), given tgBeats(lbF, lo) (the predicate holds on a prefix)
__device__ __forceinline__ int tgLastBeating(const TgInc& B, int64_t lbF, int lo, int hi) {
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (tgBeats(B, lbF, mid)) lo = mid; else hi = mid - 1;
    }
    return lo;
}

// the same by galloping from lo: for a stretch whose answer lies close to its left end (the one above the last evaluated
// threshold runs to the end of the candidate list) the probes stay inside the staged candidate window
__device__ __forceinline__ int tgLastBeatingGallop(const TgInc& B, int64_t lbF, int lo, int hi) {
    int step = 1;
    while (lo + step <= hi && tgBeats(B, lbF, lo + step)) { lo += step; step <<= 1; }
    return tgLastBeating(B, lbF, lo, min(hi, lo + step - 1));
}

__device__ void tgWriteInfeasible(const TgSolveCtx& ctx, TgInstDev& I, int i) {
    tg_result z;
    memset(&z, 0, sizeof(z));
    z.iter_time_us = INT64_MAX;
    z.n_thresholds_run = uint32_t(I.nrun);
    ctx.out[i] = z;
    I.phase = TG_PH_DONE;
}

// The previous round's items as the scheduler reads them: the first nStage are staged in shared memory by
// the whole CTA (one L2 round trip for all of them instead of one per access of a single thread).
struct TgPrev {
    const TgItem* items;
    const unsigned long long* keys;
    const unsigned long long* keyS;
    const int32_t* tidxS;
    const uint32_t* candS;   // cand[tidx] of the item's instance
    const uint8_t* flagS;
    int nStage;
    uint32_t mask;           // item index -> slot: all ones (round mode: indices of one round's array) or TG_QCAP - 1 (queue mode: ring)
    __device__ __forceinline__ int slot(int i) const { return int(uint32_t(i) & mask); }
    __device__ __forceinline__ unsigned long long key(int i) const { return i < nStage ? keyS[i] : __ldcg(keys + slot(i)); }
    __device__ __forceinline__ int tidx(int i) const { return i < nStage ? tidxS[i] : __ldcg(&items[slot(i)].tidx); }
    __device__ __forceinline__ int flags(int i) const { return i < nStage ? int(flagS[i]) : int(__ldcg(&items[slot(i)].flags)); }
    __device__ __forceinline__ uint32_t cand(const TgInstDev& I, int i, int tx) const { return i < nStage ? candS[i] : I.cand[tx]; }
};

// Fold the results of instance i's items of the previous round (ascending candidate index).
__device__ void tgFoldInstance(const TgSolveCtx& ctx, TgInstDev& I, const TgPrev& P, bool full) {
    const TgItem* itemsPrev = P.items;
    const int beg = I.itemBeg, cnt = I.itemCnt;
    I.itemCnt = 0;
    if (I.phase == TG_PH_FINAL) { I.phase = TG_PH_DONE; return; }   // result written by the back-tracker
    int nf = 0;
    int nRes = cnt;   // a speculative final DP, if any, is the last item: not a search result
    if (nRes > 0) { const int fl = P.flags(beg + nRes - 1); if ((fl & TG_IT_TRACK) && !(fl & TG_IT_ALLISL)) --nRes; }
    int loInf = I.loInf, hiFeas = I.hiFeas, incIdx = I.incIdx, incQ = -1;
    int64_t incIter = I.incIter;
    const int64_t m1 = int64_t(I.m - 1);
    unsigned long long incKey = 0;
    for (int q = 0; q < nRes; ++q) {
        const int tidx = P.tidx(beg + q);
        const unsigned long long key = P.key(beg + q);
        if (key == TG_KEY_NONE) { loInf = max(loInf, tidx); continue; }
        ++nf;
        hiFeas = hiFeas < 0 ? tidx : min(hiFeas, tidx);
        const int64_t it = int64_t(key >> 32) + m1 * int64_t(P.cand(I, beg + q, tidx));
        if (incIdx < 0 || it < incIter || (it == incIter && tidx < incIdx)) { incIter = it; incIdx = tidx; incQ = q; incKey = key; }
    }
    I.loInf = loInf; I.hiFeas = hiFeas;
    I.specItem = -1;
    if (I.specIdx >= 0)   // speculation ran: is the incumbent's back-tracked result among the items of that round?
        for (int q = 0; q < cnt; ++q)
            if ((P.flags(beg + q) & TG_IT_SPEC) && P.tidx(beg + q) == incIdx) { I.specItem = beg + q; break; }
    if (incQ >= 0) {
        I.incIter = incIter; I.incIdx = incIdx;
        const uint32_t Sc = uint32_t(incKey >> 8) & 0xffffu;   // compact labels of that item
        uint32_t So = 0;
        uint8_t isl[TG_MAX_K];   // (all 16 labels loaded at once: one L2 round trip, not one per member of the mask)
#pragma unroll
        for (int e = 0; e < TG_MAX_K; ++e) isl[e] = __ldcg(&itemsPrev[P.slot(beg + incQ)].isl[e]);
#pragma unroll
        for (int e = 0; e < TG_MAX_K; ++e) if (Sc >> e & 1u) So |= 1u << isl[e];
        I.incMask = So;
    }
    I.nrun += cnt;
    if (I.phase == TG_PH_SWEEP) { I.next = P.tidx(beg + cnt - 1) + 1; return; }
    if (nRes == 0) return;
    if (full || nf == 0) return;
    // merge the feasible results into the evaluated list (both ascending), from the back
    if (I.nEval + nf > TG_MAX_EVAL / 2) {
        // compaction: an evaluated point whose stretches on both sides are resolved is no longer needed
        // (the resolved flag of its right neighbour then covers both stretches; flags are never re-checked)
        int w = 1;
        for (int t = 1; t < I.nEval; ++t) {
            const bool last = t + 1 == I.nEval;
            const bool drop = !last && (I.eIdx[t] & TG_EDONE) && (I.eIdx[t + 1] & TG_EDONE);
            if (!drop) { I.eIdx[w] = I.eIdx[t]; I.eF[w] = I.eF[t]; ++w; }
        }
        I.nEval = min(I.nEval, w);
    }
    if (I.nEval + nf > TG_MAX_EVAL) {   // cannot happen in practice; stop the search rather than loop
        atomicExch(&ctx.ctrl->errFlag, 3);
        I.phase = TG_PH_FINAL;
        return;
    }
    const int nEval = I.nEval;
    int32_t* const eIdx = I.eIdx;
    uint32_t* const eF = I.eF;
    int e = nEval - 1, w = nEval + nf - 1, q = nRes - 1;
    while (q >= 0) {
        const unsigned long long key = P.key(beg + q);
        if (key == TG_KEY_NONE) { --q; continue; }
        const int tidx = P.tidx(beg + q);
        const int ev = e >= 0 ? eIdx[e] : 0;
        if (e >= 0 && (ev & ~TG_EDONE) > tidx) { eIdx[w] = ev; eF[w] = eF[e]; --e; --w; }
        else { eIdx[w] = tidx; eF[w] = uint32_t(key >> 32); --w; --q; }
    }
    I.nEval = nEval + nf;
}

// Plan the probes of instance i for this round into I.probe[0..nProbe).  Returns the item kind.
__device__ int tgPlanInstance(const TgSolveCtx& ctx, TgInstDev& I, int i, int W, bool full) {
    const int n = I.ncand;
    I.nProbe = 0;
    const int specItem = I.specItem;   // refers to the round just folded
    I.specItem = -1;
    if (I.phase == TG_PH_NEW) {
        if (ctx.mode == 1) I.phase = TG_PH_FINAL;
        else if (n == 0 || I.lbIdx >= n) { tgWriteInfeasible(ctx, I, i); return TG_PH_DONE; }
        else if (full) { I.phase = TG_PH_SWEEP; I.next = 0; }
        else { I.phase = TG_PH_FEAS; I.loInf = I.lbIdx - 1; I.hiFeas = -1; I.gstep = 1; }
    }
    if (I.phase == TG_PH_FEAS) {
        if (I.hiFeas < 0) {
            if (I.loInf >= n - 1) { tgWriteInfeasible(ctx, I, i); return TG_PH_DONE; }
            // galloping: loInf + gstep, + 2 gstep, ... ; at most gallopMax (10) probes a round, the step keeps doubling.
            // (More probes reach thresholds far above the optimum, whose DPs have full-width rows: 16 probes made
            // cfg3 four times slower; fewer need another round: 8 cost cfg3 20 %.)
            int step = I.gstep;
            const int nmax = min(W, ctx.gallopMax);
            while (I.nProbe < nmax) {
                const int c = min(int64_t(n - 1), int64_t(I.loInf) + step);
                I.probe[I.nProbe++] = c;
                if (c == n - 1) break;
                step = step < (1 << 28) ? step * 2 : step;
            }
            I.gstep = step;
            return TG_PH_FEAS;
        }
        const int span = I.hiFeas - I.loInf - 1;   // undecided candidates strictly inside the bracket
        if (span > 0) {
            if (span <= W) for (int q = 0; q < span; ++q) I.probe[I.nProbe++] = I.loInf + 1 + q;
            else for (int q = 0; q < W; ++q) I.probe[I.nProbe++] = I.loInf + int((int64_t(q + 1) * (span + 1)) / (W + 1));
            return TG_PH_FEAS;
        }
        I.phase = TG_PH_BNB;   // hiFeas is the lowest feasible candidate
    }
    if (I.phase == TG_PH_BNB) {
        // unresolved stretches (left end exclusive, right end inclusive), at most 16 a round
        int sLo[16], sHi[16], ns = 0;
        long long total = 0;
        bool truncated = false;
        const TgInc B = {I.incIter, int64_t(I.m - 1), I.incIdx, I.cand, I.candWin, I.candWinLo, I.candWin ? I.candWinN : 0};
        const int nEval = I.nEval;
        int32_t* const eIdx = I.eIdx;
        const uint32_t* const eF = I.eF;
        int a = eIdx[0] & ~TG_EDONE;   // left neighbour of the point under test
        for (int t = 1; t < nEval; ++t) {
            if (ns >= 15) { truncated = true; break; }
            const int ej = eIdx[t], aPrev = a;
            a = ej & ~TG_EDONE;
            if (ej & TG_EDONE) continue;
            const int64_t f = int64_t(eF[t]);
            if (ej - aPrev <= 1 || !tgBeats(B, f, aPrev + 1)) { eIdx[t] = ej | TG_EDONE; continue; }
            sLo[ns] = aPrev; sHi[ns] = tgLastBeating(B, f, aPrev + 1, ej - 1);
            total += sHi[ns] - sLo[ns];
            ++ns;
        }
        int topEnd = -1;
        {   // above the last evaluated point only the trivial bound f >= 0 is known: probe just the right end of
            // that stretch; once it is evaluated the stretch gets a real bound and shrinks
            const int last = eIdx[nEval - 1] & ~TG_EDONE;
            if (last < n - 1 && tgBeats(B, 0, last + 1)) topEnd = tgLastBeatingGallop(B, 0, last + 1, n - 1);
        }
        if (ns == 0 && topEnd < 0) I.phase = TG_PH_FINAL;
        else {
            int budget = topEnd >= 0 ? W - 1 : W;
            const int budget0 = budget;
            int32_t* const probe = I.probe;
            int np = 0;
            for (int s = 0; s < ns && budget > 0; ++s) {
                // (32-bit arithmetic: stretch sizes are counts of candidates, at most NS * K = 33 280, probes at most 64 -- a
                // 64-bit division is a ~300-cycle chain and this code is on the critical path of every round)
                const int size = sHi[s] - sLo[s];
                int share = int(max(1u, uint32_t(budget0) * uint32_t(size) / uint32_t(max(total, 1ll))));
                share = min(min(share, size), budget);
                for (int q = 1; q <= share; ++q) probe[np++] = sLo[s] + int((uint32_t(q) * uint32_t(size) + uint32_t(share - 1)) / uint32_t(share));
                budget -= share;
            }
            if (topEnd >= 0) { probe[np++] = topEnd; total += W; }   // (total += W: not every candidate is probed)
            // every unresolved candidate is probed this round: run the final DP at the incumbent alongside
            // (speculation: it stands unless one of these probes takes the incumbent over)
            int spec = -1;
            if (!truncated && total < W && np == int(total)) {
                // last round of the search.  With few instances a round costs a DP's latency whatever it holds, so
                // every probe keeps its levels and back-tracks too: whichever ends up as the optimum already has its plan
                if (ctx.nInst <= TG_SPEC_ALL_MAX_INST)
                    for (int q = 0; q < np; ++q) probe[q] |= TG_PROBE_KEEP;
                probe[np++] = B.incIdx | TG_PROBE_FINAL;
                spec = B.incIdx;
            }
            I.specIdx = spec;
            I.nProbe = np;
            return TG_PH_BNB;
        }
    }
    if (I.phase == TG_PH_SWEEP) {
        if (I.next >= n) {
            if (I.incIdx < 0) { tgWriteInfeasible(ctx, I, i); return TG_PH_DONE; }
            I.phase = TG_PH_FINAL;
        } else {
            for (int q = 0; q < W && I.next + q < n; ++q) I.probe[I.nProbe++] = I.next + q;
            return TG_PH_SWEEP;
        }
    }
    if (I.phase == TG_PH_FINAL) {
        if (ctx.mode == 0 && specItem >= 0) {   // already back-tracked (speculatively) in the round just folded
            const unsigned long long* src = reinterpret_cast<const unsigned long long*>(ctx.specOut + (specItem & (TG_QCAP - 1)));
            unsigned long long* dst = reinterpret_cast<unsigned long long*>(ctx.out + i);
            for (int w = 0; w < int(sizeof(tg_result) / 8); ++w) dst[w] = __ldcg(src + w);
            ctx.out[i].n_thresholds_run = uint32_t(I.nrun);
            I.phase = TG_PH_DONE;
            return TG_PH_DONE;
        }
        I.probe[0] = ctx.mode == 1 ? -1 : I.incIdx; I.nProbe = 1;
        return TG_PH_FINAL;
    }
    return TG_PH_DONE;
}

// Fold the previous round into every instance's search state and plan its next probes (I.probe, I.nProbe,
// I.planKind).  Narrow (few instances): CTA 0, one thread per instance, the previous items staged in shared
// memory.  Wide (many instances): the fold and the planning are single-thread, branchy code -- packed 32 to a warp
// on CTA 0 they serialise (cfg5: 0.35 ms a round with the whole grid waiting) -- so every warp of the grid takes
// at most one instance at a time (lane 0), followed by one grid barrier before CTA 0 lays the items out.
#define TG_WIDE_MIN_INST 64
__device__ void tgFoldPlanAll(const TgSolveCtx& ctx, TgShared& sm, uint32_t* dyn, int round, bool wide) {
    const int tid = threadIdx.x, prv = (round & 1) ^ 1;
    TgCtrl* ctrl = ctx.ctrl;
    const TgItem* itemsPrev = ctx.items + size_t(prv) * TG_MAX_ITEMS;
    const unsigned long long* keysPrev = ctx.keys + size_t(prv) * TG_MAX_ITEMS;
    const bool full = (ctx.flags & TG_SOLVE_FULL_SWEEP) != 0;
    if (tid == 0 && round < 8 && blockIdx.x == 0) ctrl->schedCyc[round][0] = clock64();
    TgPrev P;
    P.items = itemsPrev; P.keys = keysPrev; P.keyS = nullptr; P.tidxS = nullptr; P.candS = nullptr; P.flagS = nullptr; P.nStage = 0;
    P.mask = 0xffffffffu;
    if (!wide) {   // stage keys, candidate indices, their thresholds and flags of the previous items in the (idle) dynamic shared memory
        const int nPrev = round > 0 ? ctrl->nItems[prv] : 0;
        const int room = int(size_t(ctx.dynWords) * 4 / 20);   // 17 bytes an item, padded
        const int nStage = min(nPrev, room) & ~1;   // even: keeps the arrays behind the keys 8-byte aligned
        unsigned long long* keyS = reinterpret_cast<unsigned long long*>(dyn);
        int32_t* tidxS = reinterpret_cast<int32_t*>(keyS + nStage);
        uint32_t* candS = reinterpret_cast<uint32_t*>(tidxS + nStage);
        uint8_t* flagS = reinterpret_cast<uint8_t*>(candS + nStage);
        for (int q = tid; q < nStage; q += TG_NT) {
            const int tx = __ldcg(&itemsPrev[q].tidx);
            keyS[q] = __ldcg(keysPrev + q);
            tidxS[q] = tx;
            flagS[q] = __ldcg(&itemsPrev[q].flags);
            candS[q] = tx >= 0 ? ctx.inst[__ldcg(&itemsPrev[q].inst)].cand[tx] : 0u;
        }
        P.keyS = keyS; P.tidxS = tidxS; P.candS = candS; P.flagS = flagS; P.nStage = nStage;
        __syncthreads();
    }
    if (tid == 0 && round < 8 && blockIdx.x == 0) ctrl->dbgCyc[round][0] = clock64();
    // W is bounded by the item list shared among the instances still running (count of the previous round: an upper bound)
    const int nActive = round > 0 ? max(1, __ldcg(&ctrl->nActive)) : ctx.nInst;
    const int capAll = max(1, min(ctx.wishMax, TG_MAX_ITEMS / nActive));
    const bool mine = wide ? (tid & 31) == 0 : true;
    const int first = wide ? int(blockIdx.x) * TG_NW + (tid >> 5) : tid;
    const int stride = wide ? int(gridDim.x) * TG_NW : TG_NT;
    // A handful of instances (the latency-bound case): their search state -- the TgInstDev record and the evaluated
    // list -- is copied to shared memory by the whole CTA, folded and planned there by one thread each, and copied
    // back.  In global memory every field access of that single thread is a dependent L1/L2 access, and a store
    // invalidates the line the next load wants (the merge of the evaluated list paid one L2 trip per entry).
    constexpr int INST_W = int(sizeof(TgInstDev) / 4);
    const size_t dynWords = size_t(ctx.dynWords);
    const bool local = !wide && ctx.nInst <= TG_SCHED_SMEM_INST &&
                       ((5 * size_t(P.nStage) + 3) & ~size_t(3)) + size_t(ctx.nInst) * (INST_W + 2 * TG_MAX_EVAL + TG_CAND_WIN) <= dynWords;
    uint32_t* sInst = dyn + ((5 * size_t(P.nStage) + 3) & ~size_t(3));   // behind the staged previous items (17 bytes each)
    uint32_t* sEval = sInst + size_t(ctx.nInst) * INST_W;                 // [nInst][2][TG_MAX_EVAL]
    if (local) {
        for (int i = 0; i < ctx.nInst; ++i) {
            const uint32_t* src = reinterpret_cast<const uint32_t*>(ctx.inst + i);
            for (int w = tid; w < INST_W; w += TG_NT) sInst[size_t(i) * INST_W + w] = src[w];
        }
        __syncthreads();
        for (int i = 0; i < ctx.nInst; ++i) {
            const TgInstDev& S = *reinterpret_cast<const TgInstDev*>(sInst + size_t(i) * INST_W);
            const int ne = min(max(S.nEval, 0), TG_MAX_EVAL);
            for (int w = tid; w < ne; w += TG_NT) {
                sEval[(size_t(i) * 2 + 0) * TG_MAX_EVAL + w] = uint32_t(S.eIdx[w]);
                sEval[(size_t(i) * 2 + 1) * TG_MAX_EVAL + w] = S.eF[w];
            }
            // the candidates the bound tests will look at start at the lowest feasible one (first evaluated point)
            const int lo = ne > 0 ? int(uint32_t(S.eIdx[0]) & ~uint32_t(TG_EDONE)) : max(S.lbIdx, 0);
            const int nw = max(0, min(TG_CAND_WIN, S.ncand - lo));
            uint32_t* sCand = sEval + size_t(ctx.nInst) * 2 * TG_MAX_EVAL + size_t(i) * TG_CAND_WIN;
            tgCopyToShared(sCand, S.cand + lo, nw);   // (cand is read-only during the solve)
            if (tid == 0) {
                TgInstDev& Sw = *reinterpret_cast<TgInstDev*>(sInst + size_t(i) * INST_W);
                Sw.candWin = sCand; Sw.candWinLo = lo; Sw.candWinN = nw;
            }
        }
        __syncthreads();
    }
    if (tid == 0 && round < 8 && blockIdx.x == 0) ctrl->dbgCyc[round][1] = clock64();
    if (mine)
        for (int i = first; i < ctx.nInst; i += stride) {
            TgInstDev& I = local ? *reinterpret_cast<TgInstDev*>(sInst + size_t(i) * INST_W) : ctx.inst[i];
            int32_t* gIdx = I.eIdx;
            uint32_t* gF = I.eF;
            if (local) {
                I.eIdx = reinterpret_cast<int32_t*>(sEval + (size_t(i) * 2 + 0) * TG_MAX_EVAL);
                I.eF = sEval + (size_t(i) * 2 + 1) * TG_MAX_EVAL;
            }
            if (I.itemCnt > 0) tgFoldInstance(ctx, I, P, full);
            if (tid == 0 && round < 8 && blockIdx.x == 0) ctrl->dbgCyc[round][2] = clock64();
            if (I.phase != TG_PH_DONE) I.planKind = tgPlanInstance(ctx, I, i, full ? capAll : min(capAll, tgWish(ctx, I.K)), full);   // a full sweep has no speculation
            if (local) { I.eIdx = gIdx; I.eF = gF; I.candWin = nullptr; I.candWinN = 0; }
            if (tid == 0 && round < 8 && blockIdx.x == 0) ctrl->dbgCyc[round][3] = clock64();
        }
    __syncthreads();
    if (local) {
        for (int i = 0; i < ctx.nInst; ++i) {
            const TgInstDev& S = *reinterpret_cast<const TgInstDev*>(sInst + size_t(i) * INST_W);
            const int ne = min(max(S.nEval, 0), TG_MAX_EVAL);
            for (int w = tid; w < ne; w += TG_NT) {
                S.eIdx[w] = int32_t(sEval[(size_t(i) * 2 + 0) * TG_MAX_EVAL + w]);
                S.eF[w] = sEval[(size_t(i) * 2 + 1) * TG_MAX_EVAL + w];
            }
            uint32_t* dst = reinterpret_cast<uint32_t*>(ctx.inst + i);
            for (int w = tid; w < INST_W; w += TG_NT) dst[w] = sInst[size_t(i) * INST_W + w];
        }
        __syncthreads();
    }
    if (tid == 0 && round < 8 && blockIdx.x == 0) ctrl->schedCyc[round][1] = clock64();
}

// ---------------------------------------------------------------------------------------------
// Queue mode (a batch of TG_WIDE_MIN_INST .. TG_QUEUE_MAX_INST instances, default search).  The scheduler rounds cost
// such a batch a grid barrier per round with the whole grid waiting for the round's last DP, the slowest instance's fold
// and plan and the item layout (12 rounds: 13.5 % of the CTA cycles at cfg5, 18 % of the warp samples at the barrier).  But
// an instance's next probes depend only on its OWN results.  So after the first round is laid out the items form one
// queue in a ring of TG_QCAP slots: a CTA takes the next sequence number, waits until that item is published, runs the
// DP, and decrements its instance's count of running items; the CTA that takes it to zero folds and plans THAT instance
// right away (state machine of tgFoldInstance / tgPlanInstance, unchanged, on a shared-memory copy of the instance's
// search state) and appends its new items to the queue.  No grid barrier after the first round; CTAs leave when every
// instance is done.  An instance plans few probes at a time (TG_QUEUE_WISH, default 6) while the queue is long and the full
// width once CTAs would otherwise wait, so the NUMBER of DPs an instance runs (n_thresholds_run, a diagnostic) depends on
// the timing; the result does not -- every schedule of the exact search returns the same optimum and plan.
// Measured at cfg5: 27.8 -> 23.8 ms, 47 588 -> ~44 600 DPs, grid-wait share of the CTA cycles 13.5 -> 4 %.
// ---------------------------------------------------------------------------------------------
__device__ void tgQueueFoldPlan(const TgSolveCtx& ctx, TgShared& sm, uint32_t* dyn, int i) {
    const int tid = threadIdx.x;
    TgCtrl* ctrl = ctx.ctrl;
    constexpr int INST_W = int(sizeof(TgInstDev) / 4);
    uint32_t* sInst = dyn;                                  // [INST_W] copy of the instance record
    uint32_t* sEval = sInst + ((INST_W + 3) & ~3);          // [2][TG_MAX_EVAL] evaluated thresholds
    uint32_t* sCand = sEval + 2 * TG_MAX_EVAL;              // [TG_CAND_WIN] window of the candidate list
    __threadfence();                                        // the keys the other CTAs posted for this instance's items
    {
        const uint32_t* src = reinterpret_cast<const uint32_t*>(ctx.inst + i);
        for (int w = tid; w < INST_W; w += TG_NT) sInst[w] = __ldcg(src + w);
    }
    __syncthreads();
    TgInstDev& I = *reinterpret_cast<TgInstDev*>(sInst);
    int32_t* const gIdx = I.eIdx;
    uint32_t* const gF = I.eF;
    const int ne = min(max(I.nEval, 0), TG_MAX_EVAL);
    for (int w = tid; w < ne; w += TG_NT) { sEval[w] = uint32_t(__ldcg(gIdx + w)); sEval[TG_MAX_EVAL + w] = __ldcg(gF + w); }
    const int lo = ne > 0 ? int(uint32_t(__ldcg(gIdx)) & ~uint32_t(TG_EDONE)) : max(I.lbIdx, 0);
    const int nw = max(0, min(TG_CAND_WIN, I.ncand - lo));
    tgCopyToShared(sCand, I.cand + lo, nw);   // (cand is read-only during the solve)
    __syncthreads();
    if (tid == 0) {
        I.eIdx = reinterpret_cast<int32_t*>(sEval);
        I.eF = sEval + TG_MAX_EVAL;
        I.candWin = sCand; I.candWinLo = lo; I.candWinN = nw;
        TgPrev P;
        P.items = ctx.items; P.keys = ctx.keys; P.keyS = nullptr; P.tidxS = nullptr; P.candS = nullptr; P.flagS = nullptr;
        P.nStage = 0; P.mask = TG_QCAP - 1;
        for (int q = 0; q < I.itemCnt; ++q)   // every slot to fold still holds this instance's item (the ring did not wrap onto it)
            if (__ldcg(&ctx.items[uint32_t(I.itemBeg + q) & (TG_QCAP - 1)].seq) != uint32_t(I.itemBeg + q)) atomicExch(&ctrl->errFlag, 4);
        if (I.itemCnt > 0) tgFoldInstance(ctx, I, P, false);
        if (I.phase != TG_PH_DONE) {
            // few probes at a time while the queue is long (less speculation: an extra "round" costs this instance latency only),
            // the full width once CTAs would otherwise wait for work (the tail of the batch is bound by the instances' chains)
            const int backlog = int(__ldcg(&ctrl->qTail) - __ldcg(&ctrl->qHead));
            const int W = backlog < int(gridDim.x) ? ctx.wishCap : ctx.queueWish;
            I.planKind = tgPlanInstance(ctx, I, i, min(min(ctx.wishMax, W), max(tgWish(ctx, I.K), W)), false);
        }
        I.eIdx = gIdx; I.eF = gF; I.candWin = nullptr; I.candWinN = 0;
        int cnt = I.phase != TG_PH_DONE ? I.nProbe : 0;
        uint32_t base = 0;
        if (cnt > 0) base = atomicAdd(&ctrl->qTail, uint32_t(cnt));
        I.itemBeg = int(base); I.itemCnt = cnt; I.pending = cnt;
        sm.iTmp[3] = cnt; sm.iTmp[4] = int(base);
    }
    __syncthreads();
    {   // the record and the evaluated list go back before the new items can be seen
        const int ne2 = min(max(I.nEval, 0), TG_MAX_EVAL);
        for (int w = tid; w < ne2; w += TG_NT) { gIdx[w] = int32_t(sEval[w]); gF[w] = sEval[TG_MAX_EVAL + w]; }
        uint32_t* dst = reinterpret_cast<uint32_t*>(ctx.inst + i);
        for (int w = tid; w < INST_W; w += TG_NT) dst[w] = sInst[w];
    }
    __syncthreads();
    const int cnt = sm.iTmp[3];
    const uint32_t base = uint32_t(sm.iTmp[4]);
    if (tid < cnt) {
        const uint32_t seq = base + uint32_t(tid), slot = seq & (TG_QCAP - 1);
        TgItem& it = ctx.items[slot];
        const int kind = I.planKind, pq = I.probe[tid];
        it.inst = i;
        it.seq = seq;
        it.tidx = pq >= 0 ? (pq & ~(TG_PROBE_FINAL | TG_PROBE_KEEP)) : -1;
        it.T = it.tidx >= 0 ? I.cand[it.tidx] : ctx.dpT;
        it.flags = kind == TG_PH_FINAL ? TG_IT_TRACK
                   : (pq >= 0 && (pq & TG_PROBE_FINAL)) ? (TG_IT_TRACK | TG_IT_SPEC)
                   : (pq >= 0 && (pq & TG_PROBE_KEEP)) ? (TG_IT_TRACK | TG_IT_SPEC | TG_IT_ALLISL) : 0;
        ctx.keys[slot] = TG_KEY_NONE;
        __threadfence();
        asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(ctx.itemSeq + slot), "r"(seq + 1u) : "memory");
    }
    if (tid == 0) {
        if (cnt > 0) atomicAdd((unsigned long long*)&ctrl->stats.n_dp, (unsigned long long)cnt);
        else {   // the instance is finished (its result was written by the back-tracker or while planning)
            const int d = atomicAdd(&ctrl->nDoneInst, 1) + 1;
            if (d == ctx.nInst) { __threadfence(); atomicExch(&ctrl->allDone, 1); }
        }
    }
    __syncthreads();
}

// Scheduler, second half (CTA 0): lay the planned probes out as the round's item list, size the teams.
__device__ void tgSchedule(const TgSolveCtx& ctx, TgShared& sm, int round) {
    const int tid = threadIdx.x;
    const int par = round & 1;
    TgCtrl* ctrl = ctx.ctrl;
    TgItem* items = ctx.items + size_t(par) * TG_MAX_ITEMS;
    unsigned long long* keys = ctx.keys + size_t(par) * TG_MAX_ITEMS;
    const int nInst = ctx.nInst;

    if (tid == 0) { sm.iTmp[0] = 0; sm.iTmp[1] = 0; sm.llTmp[0] = 0; sm.llTmp[1] = 0; }
    __syncthreads();
    int nActive = 0;
    for (int i = tid; i < nInst; i += TG_NT) nActive += ctx.inst[i].phase != TG_PH_DONE ? 1 : 0;
    if (nActive) atomicAdd(&sm.iTmp[0], nActive);
    __syncthreads();
    nActive = sm.iTmp[0];
    if (nActive == 0) {
        if (tid == 0) { ctrl->done = 1; ctrl->nItems[par] = 0; }
        return;
    }
    if (tid == 0) ctrl->nActive = nActive;

    // ---- B: plan every instance's probes, lay the items out ------------------------------------------
    uint32_t carry = 0;
    for (int base = 0; base < nInst; base += TG_NT) {
        const int i = base + tid;
        int cnt = 0, kind = TG_PH_DONE;
        if (i < nInst && ctx.inst[i].phase != TG_PH_DONE) {
            TgInstDev& I = ctx.inst[i];
            kind = I.planKind;
            cnt = I.nProbe;
        }
        uint32_t tot;
        const uint32_t pos = tgBlockExScan(uint32_t(cnt), sm.warpSums, tot) + carry;
        carry += tot;
        if (cnt > 0) {
            TgInstDev& I = ctx.inst[i];
            if (pos + cnt > TG_MAX_ITEMS) { cnt = 0; I.specIdx = -1; }   // more active instances than items: wait a round
            I.itemBeg = int(pos); I.itemCnt = cnt;
            if (cnt > 0) atomicMax(&sm.iTmp[1], int(pos) + cnt);
            if (nInst > TG_NW)   // many instances: one thread lays out its instance's probes (a handful: below)
            for (int q = 0; q < cnt; ++q) {
                TgItem& it = items[pos + q];
                it.inst = i;
                const int pq = I.probe[q];
                it.tidx = pq >= 0 ? (pq & ~(TG_PROBE_FINAL | TG_PROBE_KEEP)) : -1;
                it.T = it.tidx >= 0 ? I.cand[it.tidx] : ctx.dpT;
                it.flags = kind == TG_PH_FINAL ? TG_IT_TRACK
                           : (pq >= 0 && (pq & TG_PROBE_FINAL)) ? (TG_IT_TRACK | TG_IT_SPEC)
                           : (pq >= 0 && (pq & TG_PROBE_KEEP)) ? (TG_IT_TRACK | TG_IT_SPEC | TG_IT_ALLISL) : 0;
            }
        }
    }
    __syncthreads();
    if (nInst <= TG_NW) {
        // a handful of instances (the latency-bound case): warp w lays out instance w's probes, one lane per probe -- the
        // chain probe -> candidate threshold -> item is two dependent L2 round trips, paid once instead of once per probe
        const int w = tid >> 5, lane = tid & 31;
        if (w < nInst && ctx.inst[w].phase != TG_PH_DONE) {
            TgInstDev& I = ctx.inst[w];
            const int cnt = I.itemCnt, pos = I.itemBeg, kind = I.planKind;
            for (int q = lane; q < cnt; q += 32) {
                TgItem& it = items[pos + q];
                it.inst = w;
                const int pq = I.probe[q];
                it.tidx = pq >= 0 ? (pq & ~(TG_PROBE_FINAL | TG_PROBE_KEEP)) : -1;
                it.T = it.tidx >= 0 ? I.cand[it.tidx] : ctx.dpT;
                it.flags = kind == TG_PH_FINAL ? TG_IT_TRACK
                           : (pq >= 0 && (pq & TG_PROBE_FINAL)) ? (TG_IT_TRACK | TG_IT_SPEC)
                           : (pq >= 0 && (pq & TG_PROBE_KEEP)) ? (TG_IT_TRACK | TG_IT_SPEC | TG_IT_ALLISL) : 0;
            }
        }
        __syncthreads();
    }
    const int nIt = sm.iTmp[1];
    if (tid == 0 && round < 8) ctrl->schedCyc[round][2] = clock64();

    // (the geometry of an item -- islands alive at its T -- is worked out by the CTAs that run it)
    for (int idx = tid; idx < nIt; idx += TG_NT) keys[idx] = TG_KEY_NONE;
    for (int s = tid; s < ctx.nSlots; s += TG_NT) ctx.slotBar[s] = 0;
    __syncthreads();
    // ---- C: team sizes.  A few items share the grid as teams of CTAs; a DP's cost varies a lot with its
    // threshold (row-window width, islands alive) and with the instance shape, so the CTAs are dealt out in
    // proportion to an estimate of it:  masks x rows x (per-row bookkeeping + lanes a row's chunks occupy).
    const bool weighted = nIt > 1 && nIt <= 32 && nIt < ctx.nSlots && gridDim.x <= 1024;
    if (weighted) {
        const int lane = tid & 31, warp = tid >> 5;
        for (int t = warp; t < nIt; t += TG_NW) {
            const TgItem& it = items[t];
            const TgInstDev& I = ctx.inst[it.inst];
            const int L = I.L, K = I.K;
            const uint32_t T = it.T;
            const uint32_t allow = ((it.flags & TG_IT_TRACK) && !(it.flags & TG_IT_ALLISL) && ctx.mode == 0) ? I.incMask : 0xffffu;   // as in tgStageItem
            // lane = (island k, half of the lengths d): counts the admissible lengths of its half -- sufMinAll is
            // non-decreasing in d, so the count over both halves is the longest admissible slice of k
            const int k = lane & 15, half = lane >> 4;
            unsigned cnt = 0;
            if (k < K && (allow >> k & 1u)) {
                const uint32_t* sf = I.sufMinAll + size_t(k) * (L + 2);
#pragma unroll 32
                for (int d = 1 + half; d <= L; d += 2) cnt += (sf[d] <= T) ? 1u : 0u;
            }
            cnt += __shfl_xor_sync(0xffffffffu, cnt, 16);
            const int ke = __popc(__ballot_sync(0xffffffffu, cnt > 0) & 0xffffu);
            const int ctot = int(__reduce_add_sync(0xffffffffu, half == 0 ? cnt : 0u));
            if (lane == 0) {
                float w = 1.0f;
                if (ctot >= L && ke > 0) {
                    const int wd = min(I.Lp, (ctot - L + 4 + 3) & ~3), nbw = wd >> 2;
                    int chp = 2;
                    while (chp < nbw && chp < 16) chp <<= 1;
                    w = float(ke) * exp2f(float(ke - 1)) * (3.5f + float(max(chp, nbw)));
                    if (it.flags & 1) w *= 1.5f;   // every level kept, a back-track at the end
                }
                sm.wgt[t] = w;
            }
        }
        __syncthreads();
        if (tid < 32) {
            const int nCta = int(gridDim.x);
            const float w = tid < nIt ? sm.wgt[tid] : 0.0f;
            float tot = w;
            for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
            int n = tid < nIt ? max(1, int(w / tot * float(nCta))) : 0;
            int used = int(__reduce_add_sync(0xffffffffu, unsigned(n)));
            // hand out what the rounding left (or take back what the one-CTA minimum overdrew), one CTA at a time,
            // where it changes the slowest team's estimated time the most (least)
            for (int guard = 0; used != nCta && guard < 512; ++guard) {
                const bool give = used < nCta;
                float v = tid < nIt ? (give ? w / float(n) : (n > 1 ? -w / float(n - 1) : -3.0e38f)) : -3.4e38f;
                int who = tid;
                for (int o = 16; o > 0; o >>= 1) {
                    const float ov = __shfl_xor_sync(0xffffffffu, v, o);
                    const int ow = __shfl_xor_sync(0xffffffffu, who, o);
                    if (ov > v || (ov == v && ow < who)) { v = ov; who = ow; }
                }
                if (tid == who) n += give ? 1 : -1;
                used += give ? 1 : -1;
            }
            int beg = n;
            for (int o = 1; o < 32; o <<= 1) {
                const int a = __shfl_up_sync(0xffffffffu, beg, o);
                if (tid >= o) beg += a;
            }
            beg -= n;
            if (tid < nIt) {
                items[tid].ctaBeg = uint16_t(beg);
                items[tid].ctaCnt = uint16_t(n);
                for (int c = beg; c < beg + n; ++c) ctrl->teamOf[par][c] = uint8_t(tid);
            }
        }
        __syncthreads();
    }
    if (tid == 0) {
        ctrl->weighted[par] = weighted ? 1 : 0;
        if (round < 8) ctrl->schedCyc[round][3] = clock64();
        if (round < 256) {
            unsigned long long ns;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(ns));
            ctrl->roundNs[round] = ns;
            ctrl->roundItems[round] = nIt;
        }
        ctrl->nItems[par] = nIt;
        ctrl->queue[par] = 0;
        ctrl->stats.n_dp += uint64_t(nIt);
        ctrl->stats.n_rounds += 1;
        if (nIt == 0) ctrl->done = 1;   // every remaining instance was found infeasible while planning
    }
}

// ---------------------------------------------------------------------------------------------
// The persistent kernel
// ---------------------------------------------------------------------------------------------
extern __shared__ uint4 tgDynSmem[];

__global__ void __launch_bounds__(TG_NT, TG_CTAS_PER_SM) tgSolveKernel(const TgSolveCtx ctx) {
    __shared__ TgShared sm;
    uint32_t* dyn = reinterpret_cast<uint32_t*>(tgDynSmem);
    uint32_t* Cs = dyn;
    uint32_t* wbufAll = dyn;   // the split between cost rows and warp buffers is per item (tgStageItem)
    uint32_t epoch = 0;
    TgCtrl* ctrl = ctx.ctrl;
    const int nCta = int(gridDim.x), b = int(blockIdx.x);
    if (threadIdx.x == 0) {
        for (int i = 0; i < 8; ++i) sm.cyc[i] = 0;
        sm.tmark = clock64();
    }
    for (int w = threadIdx.x; w < 17 * 17; w += TG_NT) sm.binom[w / 17][w % 17] = tgBinom[w / 17][w % 17];
    if (threadIdx.x < TG_MAX_K) sm.xInf[threadIdx.x] = TG_INFU;
#if TG_STAGE_TMA
    if (threadIdx.x == 0) {
        sm.mbarPhase = 0;
        asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(tgSmemAddr(&sm.mbar)), "r"(TG_NT) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
#endif
    __syncthreads();
    const bool wide = ctx.nInst >= TG_WIDE_MIN_INST;
    const bool queue = wide && ctx.nInst <= TG_QUEUE_MAX_INST && ctx.mode == 0 && !(ctx.flags & TG_SOLVE_FULL_SWEEP);
    if (queue) {
        // first round as in round mode (every warp of the grid plans at most one instance at a time, CTA 0 lays the items
        // out), then the queue
        tgFoldPlanAll(ctx, sm, dyn, 0, true);
        tgMark(sm, 6);
        tgGridBarrier(ctrl, epoch);
        if (b == 0) {
            tgSchedule(ctx, sm, 0);
            __syncthreads();
            const int nIt = ctrl->nItems[0];
            for (int q = threadIdx.x; q < nIt; q += TG_NT) { ctx.items[q].seq = uint32_t(q); ctx.itemSeq[q] = uint32_t(q) + 1u; }
            int done = 0;
            for (int i = threadIdx.x; i < ctx.nInst; i += TG_NT) {
                TgInstDev& I = ctx.inst[i];
                I.pending = I.itemCnt;
                if (I.phase == TG_PH_DONE || I.itemCnt == 0) { ++done; I.phase = TG_PH_DONE; }
            }
            if (done) atomicAdd(&ctrl->nDoneInst, done);
            __syncthreads();
            if (threadIdx.x == 0) {
                ctrl->qTail = uint32_t(nIt);
                if (ctrl->nDoneInst >= ctx.nInst) ctrl->allDone = 1;
            }
            tgMark(sm, 6);
        }
        tgGridBarrier(ctrl, epoch);
        tgMark(sm, 5);
        // (thread 0) the ticket after the current one is taken while the current item runs, as long as the queue is long: the
        // two L2 round trips of a fetch (ticket, publication flag) then overlap the DP.  On a short queue an early ticket
        // would hold an item back that an idle CTA could run, so there the ticket is taken when it is needed.
        uint32_t nextSeq = 0;
        bool haveNext = false;
        while (true) {
            __syncthreads();
            if (threadIdx.x == 0) {
                const uint32_t seq = haveNext ? nextSeq : atomicAdd(&ctrl->qHead, 1u);
                haveNext = false;
                if (int(__ldcg(&ctrl->qTail) - seq) > 2 * int(gridDim.x)) { nextSeq = atomicAdd(&ctrl->qHead, 1u); haveNext = true; }
                const uint32_t* flag = ctx.itemSeq + (seq & (TG_QCAP - 1));
                int got = 1;
                const long long t0 = clock64();
                while (true) {
                    uint32_t v;
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(flag) : "memory");
                    if (v == seq + 1u) break;
                    int dn;
                    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(dn) : "l"(&ctrl->allDone) : "memory");
                    if (dn) { got = 0; break; }
                    if (clock64() - t0 > 40000000000ll) {   // ~20 s without a new item and without the end: a lost item; stop, do not hang
                        atomicExch(&ctrl->errFlag, 5);
                        atomicExch(&ctrl->allDone, 1);
                        got = 0;
                        break;
                    }
                    __nanosleep(100);
                }
                sm.curItem = got ? int(seq) : -1;
            }
            __syncthreads();
            tgMark(sm, 5);
            const int seq = sm.curItem;
            if (seq < 0) break;
            const int slot = seq & (TG_QCAP - 1);
            tgRunItem(ctx, sm, Cs, wbufAll, ctx.items + slot, ctx.keys + slot, 0, 1, b, slot);
            if (threadIdx.x == 0) {
                __threadfence();   // this DP's key (and, for a tracked item, its result) before the count
                const int inst = __ldcg(&ctx.items[slot].inst);
                const int left = atomicSub(&ctx.inst[inst].pending, 1) - 1;
                sm.iTmp[2] = left == 0 ? inst : -1;
            }
            __syncthreads();
            tgMark(sm, 0);
            if (sm.iTmp[2] >= 0) { tgQueueFoldPlan(ctx, sm, dyn, sm.iTmp[2]); tgMark(sm, 6); }
        }
        if (threadIdx.x == 0) {
            tg_solve_stats& S = ctrl->stats;
            atomicAdd((unsigned long long*)&S.cyc_stage, sm.cyc[0]);
            atomicAdd((unsigned long long*)&S.cyc_levels, sm.cyc[3]);
            atomicAdd((unsigned long long*)&S.cyc_level_barrier, sm.cyc[4]);
            atomicAdd((unsigned long long*)&S.cyc_grid_wait, sm.cyc[5]);
            atomicAdd((unsigned long long*)&S.cyc_scheduler, sm.cyc[6]);
            atomicAdd((unsigned long long*)&S.cyc_backtrack, sm.cyc[7]);
        }
        if (b == 0 && threadIdx.x == 0) ctrl->stats.n_barriers = epoch;
        return;
    }
    for (int round = 0;; ++round) {
        const int par = round & 1;
        if (wide || b == 0) { tgFoldPlanAll(ctx, sm, dyn, round, wide); tgMark(sm, 6); }
        if (wide) { tgGridBarrier(ctrl, epoch); tgMark(sm, 5); }
        if (b == 0) { tgSchedule(ctx, sm, round); tgMark(sm, 6); }
        tgGridBarrier(ctrl, epoch);
        tgMark(sm, 5);
        if (__ldcg(&ctrl->done)) break;
        const int nItems = __ldcg(&ctrl->nItems[par]);
        const TgItem* items = ctx.items + size_t(par) * TG_MAX_ITEMS;
        unsigned long long* keys = ctx.keys + size_t(par) * TG_MAX_ITEMS;
        if (nItems >= ctx.nSlots) {
            // solo mode: slot = CTA; whole DPs from the queue
            if (b < ctx.nSlots) {
                while (true) {
                    __syncthreads();
                    if (threadIdx.x == 0) sm.curItem = int(atomicAdd(&ctrl->queue[par], 1u));
                    __syncthreads();
                    const int it = sm.curItem;
                    if (it >= nItems) break;
                    tgRunItem(ctx, sm, Cs, wbufAll, items + it, keys + it, 0, 1, b, it);
                }
            }
        } else {
            // team mode: team t = CTAs [t*nCta/nItems, (t+1)*nCta/nItems), slot = t
            int t, start, end;
            if (__ldcg(&ctrl->weighted[par])) {   // team sizes follow the estimated cost of the items
                t = int(__ldcg(&ctrl->teamOf[par][b]));
                start = int(__ldcg(&items[t].ctaBeg));
                end = start + int(__ldcg(&items[t].ctaCnt));
            } else {
                t = int((int64_t(b) * nItems) / nCta);
                while (t + 1 < nItems && int((int64_t(t + 1) * nCta) / nItems) <= b) ++t;
                while (t > 0 && int((int64_t(t) * nCta) / nItems) > b) --t;
                start = int((int64_t(t) * nCta) / nItems);
                end = int((int64_t(t + 1) * nCta) / nItems);
            }
            tgRunItem(ctx, sm, Cs, wbufAll, items + t, keys + t, b - start, end - start, t, t);
            if (b == start && threadIdx.x == 0 && round < 8 && t < 16) {
                unsigned long long ns;
                asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(ns));
                ctrl->itemNs[round][t] = ns;
                ctrl->itemTidx[round][t] = items[t].tidx;
            }
        }
        tgMark(sm, 0);
        tgGridBarrier(ctrl, epoch);
        tgMark(sm, 5);
    }
    if (threadIdx.x == 0) {
        tg_solve_stats& S = ctrl->stats;
        atomicAdd((unsigned long long*)&S.cyc_stage, sm.cyc[0]);
        atomicAdd((unsigned long long*)&S.cyc_levels, sm.cyc[3]);
        atomicAdd((unsigned long long*)&S.cyc_level_barrier, sm.cyc[4]);
        atomicAdd((unsigned long long*)&S.cyc_grid_wait, sm.cyc[5]);
        atomicAdd((unsigned long long*)&S.cyc_scheduler, sm.cyc[6]);
        atomicAdd((unsigned long long*)&S.cyc_backtrack, sm.cyc[7]);
    }
    if (b == 0 && threadIdx.x == 0) ctrl->stats.n_barriers = epoch;
}

// Runs behind the solver on the same stream: if the solver raised its internal error flag (a back-track without a
// predecessor, an overflowing list of evaluated thresholds) every result of the call is marked unusable
// (n_stages = -1, iter_time_us = INT64_MAX), so that a caller who never synchronises on a status -- DEVICE results, no
// statistics -- cannot take a plan from a failed search for the optimum.
__global__ void tgPoisonOnErrorKernel(const TgCtrl* __restrict__ ctrl, tg_result* __restrict__ out, int n) {
    if (ctrl->errFlag == 0) return;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        out[i].n_stages = -1;
        out[i].iter_time_us = INT64_MAX;
    }
}

}  // namespace TG_SOLVE_NS
#undef TG_COST_AT
#undef TG_COST_AT4
