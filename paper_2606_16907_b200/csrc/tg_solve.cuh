// Persistent cooperative solver: scheduler state machine, per-T popcount-wavefront DP
// (SURVEY.md §8(a) steps 4-5), threshold-sweep reduction (step 6) and plan back-tracker (step 7).
//
// One launch per tg_solve_batch.  Grid = one CTA per SM (cooperative launch, all CTAs resident).
// A scheduler round is: CTA 0 folds the previous round's results into the per-instance state
// machines and plans the next list of (instance, T) DPs ("items"); then all CTAs walk the
// wavefront levels r = |R| = 0, 1, ... of ALL items of the round in lockstep, separated by a
// grid-wide barrier, because level r reads only level r-1 (PAPER.md:250 (2): a stage is added in
// front of a memoised suffix).  State g[a][S][k] is stored as G_r[rank(R)][slot(k)][a], R = S\{k}.
//
// One tile = up to 32 masks R of one level of one item, processed by one CTA:
//   phase 1  H[R][k][b] = min_{j in R} x[k][j] + G_{r-1}[R\{j}][j][b]      (transfer pre-minimum;
//            every source row is read from L2 once per tile, results stay in shared memory)
//   phase 2  G_r[R][k][a] = min_{b>a, c<=T} c_k[a][b] + H[R][k][b]         (min-plus product against
//            the thresholded, diagonal-major cost tables staged in shared memory; 4x4 register
//            tiles, one add-min (VIADDMNMX) per relaxation, only admissible diagonals visited)
#pragma once
#include "tg_common.cuh"
#include "tg_prep.cuh"

#define TG_MAXG 160           // groups of 4 pairs per tile: <= 512/4 + 16
#define TG_NP_CAP 512         // rows of the H tile, upper bound

struct TgShared {
    // staged item
    int stagedItem;           // round * TG_MAX_ITEMS + item index, -1 = nothing staged
    int useGlobalC;
    int sL, sLp, sKe, sInst;
    uint32_t sT;
    uint32_t baseK[TG_MAX_K];
    int dmaxK[TG_MAX_K];
    int dmaxTile[TG_MAX_K][64];
    uint32_t xS[TG_MAX_K][TG_MAX_K];
    uint8_t isl[TG_MAX_K];
    uint16_t rowOffS[258];
    // tile
    uint16_t tileMask[TG_MAX_NR];
    uint8_t kList[TG_MAX_NR][TG_MAX_K];
    uint8_t jList[TG_MAX_NR][TG_MAX_K];
    uint32_t srcRow[TG_MAX_NR][TG_MAX_K];
    uint16_t grpPair[TG_MAXG][4];
    uint8_t grpK[TG_MAXG];
    int nGroups;
    unsigned long long tileKey;
    // scheduler
    uint32_t warpSums[33];
    int iTmp[8];
    unsigned long long llTmp[2];
};

__device__ __forceinline__ uint32_t tgAddMin(uint32_t a, uint32_t b, uint32_t c) { return __viaddmin_u32(a, b, c); }

__device__ __forceinline__ uint4 tgLdcg4(const uint32_t* p) { return __ldcg(reinterpret_cast<const uint4*>(p)); }

// Grid-wide barrier on a monotone counter (all CTAs are co-resident: cooperative launch).
__device__ __forceinline__ void tgGridBarrier(TgCtrl* ctrl, uint32_t& epoch) {
    __syncthreads();
    if (threadIdx.x == 0) {
        ++epoch;
        __threadfence();
        atomicAdd(&ctrl->barrier, 1u);
        const uint32_t target = epoch * gridDim.x;
        while (true) {
            const uint32_t v = *reinterpret_cast<volatile uint32_t*>(&ctrl->barrier);
            if (int32_t(v - target) >= 0) break;
            __nanosleep(32);
        }
        __threadfence();
    }
    __syncthreads();
}

// rows (R,k) of wavefront level r with Ke islands alive
__device__ __forceinline__ uint32_t tgLevelRows(int Ke, int r) { return uint32_t(tgBinom[Ke][r]) * uint32_t(Ke - r); }

__device__ __forceinline__ uint64_t tgLevelOff(const TgItem& it, int Lp, int r) {
    if (it.bufWords) return it.off + uint64_t(r & 1) * it.bufWords;
    uint64_t rows = 0;
    for (int q = 0; q < r; ++q) rows += tgLevelRows(it.Ke, q);
    return it.off + rows * uint64_t(Lp);
}

// H-tile rows available for an instance of padded length Lp (one row is reserved as the all-INF dummy)
__device__ __forceinline__ int tgNP(const TgSolveCtx& ctx, int Lp) {
    return min(ctx.hsWords / (Lp + 8) - 1, TG_NP_CAP);
}
__device__ __forceinline__ int tgNR(int np, int nk) { return max(1, min(TG_MAX_NR, np / nk)); }
__device__ __forceinline__ uint32_t tgTiles(const TgSolveCtx& ctx, int Ke, int Lp, int r) {
    if (r >= Ke) return 0;
    if (r == 0) return 1;
    const int nr = tgNR(tgNP(ctx, Lp), Ke - r);
    return (uint32_t(tgBinom[Ke][r]) + nr - 1) / nr;
}

// ---------------------------------------------------------------------------------------------
// Staging of one item's thresholded cost tables into shared memory.
//   Cs_k[d][a] = c[a][a+d][k] if <= T and a+d <= L-1, else INF   (k in compact labels)
// Only diagonals d <= dmaxK[k] (widest admissible slice of island k at T) are staged; dmaxTile
// gives the widest admissible diagonal of each 4-row tile, which bounds the phase-2 loop.
// ---------------------------------------------------------------------------------------------
__device__ void tgStageItem(const TgSolveCtx& ctx, TgShared& sm, uint32_t* Cs, uint32_t* Hs, const TgItem* itp, int itemId) {
    __syncthreads();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nWarps = TG_NT >> 5;
    const TgInstDev& I = ctx.inst[__ldcg(&itp->inst)];
    const int L = I.L, Lp = I.Lp, Ke = __ldcg(&itp->Ke);
    const uint32_t T = __ldcg(&itp->T);
    if (tid == 0) { sm.stagedItem = itemId; sm.sL = L; sm.sLp = Lp; sm.sKe = Ke; sm.sT = T; sm.sInst = itp->inst; }
    if (tid < TG_MAX_K) sm.isl[tid] = __ldcg(&itp->isl[tid]);
    for (int d = tid; d <= L + 1; d += TG_NT) sm.rowOffS[d] = d >= 1 && d <= L ? uint16_t(tgSOff(L, d)) : uint16_t(0);
    if (tid < Ke * Ke) {
        const int kc = tid / Ke, jc = tid - kc * Ke;
        sm.xS[kc][jc] = I.x[int(__ldcg(&itp->isl[kc])) * TG_MAX_K + int(__ldcg(&itp->isl[jc]))];
    }
    if (tid < Ke) {  // widest diagonal with an admissible entry: sufMin is non-decreasing in d
        const uint32_t* sf = I.sufMin + size_t(__ldcg(&itp->isl[tid])) * (L + 2);
        int lo = 0, hi = L - 1;  // answer in [0, L-1]; 0 = none
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (sf[mid] <= T) lo = mid; else hi = mid - 1;
        }
        sm.dmaxK[tid] = lo;
    }
    for (int w = tid; w < TG_MAX_K * 64; w += TG_NT) (&sm.dmaxTile[0][0])[w] = 0;
    __syncthreads();
    if (tid == 0) {
        uint32_t acc = 0;
        for (int kc = 0; kc < Ke; ++kc) { sm.baseK[kc] = acc; acc += sm.rowOffS[sm.dmaxK[kc] + 1]; }
        sm.useGlobalC = acc > uint32_t(ctx.csWords) ? 1 : 0;
        if (sm.useGlobalC) atomicAdd((unsigned long long*)&ctx.ctrl->stats.n_items_global_c, 1ull);
    }
    // the all-INF dummy row of the H tile
    {
        const int HS = Lp + 8, np = tgNP(ctx, Lp);
        for (int w = tid; w < HS; w += TG_NT) Hs[np * HS + w] = TG_INFU;
    }
    __syncthreads();
    if (!sm.useGlobalC) {
        for (int kc = 0; kc < Ke; ++kc) {
            const int dk = sm.dmaxK[kc];
            const uint32_t* cdk = I.cd + size_t(sm.isl[kc]) * I.triG;
            uint32_t* dst = Cs + sm.baseK[kc];
            for (int d0 = 1 + warp * 2; d0 <= dk; d0 += nWarps * 2) {
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    const int d = d0 + u;
                    if (d > dk) break;
                    const int rl4 = (L - d + 3) >> 2;
                    const uint32_t* src = cdk + tgGOff(L, d);
                    for (int a4 = lane; a4 < rl4; a4 += 32) {
                        uint4 v = __ldg(reinterpret_cast<const uint4*>(src) + a4);
                        const int a = a4 * 4, amax = L - 1 - d;
                        v.x = (a + 0 <= amax && v.x <= T) ? v.x : TG_INFU;
                        v.y = (a + 1 <= amax && v.y <= T) ? v.y : TG_INFU;
                        v.z = (a + 2 <= amax && v.z <= T) ? v.z : TG_INFU;
                        v.w = (a + 3 <= amax && v.w <= T) ? v.w : TG_INFU;
                        reinterpret_cast<uint4*>(dst + sm.rowOffS[d])[a4] = v;
                        if (min(min(v.x, v.y), min(v.z, v.w)) < TG_INFU) atomicMax(&sm.dmaxTile[kc][a4], d);
                    }
                }
            }
        }
    }
    __syncthreads();
}

// ---------------------------------------------------------------------------------------------
// Level 0: R = {} : G_0[k][a] = c[a][L][k] if <= T  (single stage [a,L) on island k)
// ---------------------------------------------------------------------------------------------
__device__ void tgLevel0(const TgSolveCtx& ctx, TgShared& sm, const TgItem* itp, int itemIdx, unsigned long long* keys) {
    const TgInstDev& I = ctx.inst[sm.sInst];
    const int L = sm.sL, Lp = sm.sLp, Ke = sm.sKe;
    const uint32_t T = sm.sT;
    uint32_t* G = ctx.scratch + __ldcg(&itp->off);  // level 0 sits at the item's base in both layouts
    for (int w = threadIdx.x; w < Ke * Lp; w += TG_NT) {
        const int kc = w / Lp, a = w - kc * Lp;
        uint32_t v = TG_INFU;
        if (a < L) {
            v = I.cd[size_t(sm.isl[kc]) * I.triG + tgGOff(L, L - a) + a];
            if (v > T) v = TG_INFU;
        }
        G[w] = v;
        if (a == 0 && v < TG_INFU)
            atomicMin(keys + itemIdx, (unsigned long long)v << 32 | (unsigned long long)(1u << kc) << 8 | (unsigned long long)kc);
    }
}

// ---------------------------------------------------------------------------------------------
// One tile of level r >= 1: masks R = maskOf[popOff[r] + first .. first+cnt) of the staged item.
// ---------------------------------------------------------------------------------------------
__device__ void tgTile(const TgSolveCtx& ctx, TgShared& sm, const uint32_t* Cs, uint32_t* Hs, const TgItem* itp,
                       int itemIdx, unsigned long long* keys, int r, int tile) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nWarps = TG_NT >> 5;
    const TgInstDev& I = ctx.inst[sm.sInst];
    const int L = sm.sL, Lp = sm.sLp, Ke = sm.sKe, HS = Lp + 8, nb4 = Lp >> 2;
    const uint32_t T = sm.sT;
    const int nk = Ke - r;
    const int np = tgNP(ctx, Lp), NR = tgNR(np, nk);
    const int nMasks = tgBinom[Ke][r];
    const int first = tile * NR, cnt = min(NR, nMasks - first);
    TgItem itv;
    itv.off = __ldcg(&itp->off); itv.bufWords = __ldcg(&itp->bufWords); itv.Ke = uint8_t(Ke);
    const uint32_t* Gprev = ctx.scratch + tgLevelOff(itv, Lp, r - 1);
    uint32_t* Gcur = ctx.scratch + tgLevelOff(itv, Lp, r);

    // ---- phase 0: tile metadata -------------------------------------------------------------
    if (tid < cnt) {
        const uint32_t R = ctx.maskOf[tgPopOff[r] + first + tid];
        sm.tileMask[tid] = uint16_t(R);
        int ji = 0, ki = 0;
        for (int e = 0; e < Ke; ++e) {
            if (R >> e & 1u) {
                const uint32_t Rp = R ^ (1u << e);
                sm.srcRow[tid][ji] = uint32_t(ctx.rankOf[Rp]) * uint32_t(nk + 1) + uint32_t(e - __popc(R & ((1u << e) - 1u)));
                sm.jList[tid][ji++] = uint8_t(e);
            } else {
                sm.kList[tid][ki++] = uint8_t(e);
            }
        }
    }
    if (warp == 0) {
        const uint32_t R = lane < cnt ? uint32_t(ctx.maskOf[tgPopOff[r] + first + lane]) : 0xffffffffu;
        int gbase = 0;
        for (int k = 0; k < Ke; ++k) {
            const bool ex = !(R >> k & 1u);
            const uint32_t bal = __ballot_sync(0xffffffffu, ex);
            const int n = __popc(bal), ng = (n + 3) >> 2;
            if (ex) {
                const int rk = __popc(bal & ((1u << lane) - 1u));
                sm.grpPair[gbase + (rk >> 2)][rk & 3] = uint16_t(lane * nk + (k - __popc(R & ((1u << k) - 1u))));
            }
            if (lane < ng) sm.grpK[gbase + lane] = uint8_t(k);
            if (lane < ((4 - (n & 3)) & 3)) sm.grpPair[gbase + ng - 1][3 - lane] = 0xffffu;  // pad the last group
            gbase += ng;
        }
        if (lane == 0) { sm.nGroups = gbase; sm.tileKey = TG_KEY_NONE; }
    }
    __syncthreads();

    // ---- phase 1: transfer pre-minimum into the H tile ----------------------------------------
    // Hs[pair][i] = H[b = i+1]; thread = (mask, 4 consecutive b); all k not in R at once.
    for (int w = tid; w < cnt * nb4; w += TG_NT) {
        const int rl = w / nb4, b4 = w - rl * nb4;
        uint32_t acc[TG_MAX_K - 1][4];
#pragma unroll
        for (int s = 0; s < TG_MAX_K - 1; ++s) { acc[s][0] = acc[s][1] = acc[s][2] = acc[s][3] = TG_INFU; }
        for (int ji = 0; ji < r; ++ji) {
            const uint32_t* src = Gprev + size_t(sm.srcRow[rl][ji]) * Lp + 4 * b4;
            const uint4 g4 = tgLdcg4(src);
            const uint32_t nx = (b4 + 1 < nb4) ? __ldcg(src + 4) : TG_INFU;
            const uint32_t* xr = &sm.xS[0][sm.jList[rl][ji]];
#pragma unroll
            for (int s = 0; s < TG_MAX_K - 1; ++s) {
                if (s < nk) {
                    const uint32_t xv = xr[int(sm.kList[rl][s]) * TG_MAX_K];   // x[k][j]: k sends to j
                    acc[s][0] = tgAddMin(xv, g4.y, acc[s][0]);
                    acc[s][1] = tgAddMin(xv, g4.z, acc[s][1]);
                    acc[s][2] = tgAddMin(xv, g4.w, acc[s][2]);
                    acc[s][3] = tgAddMin(xv, nx, acc[s][3]);
                }
            }
        }
        uint32_t* hrow = Hs + size_t(rl * nk) * HS + 4 * b4;
#pragma unroll
        for (int s = 0; s < TG_MAX_K - 1; ++s) {
            if (s < nk) {
                *reinterpret_cast<uint4*>(hrow + size_t(s) * HS) = make_uint4(acc[s][0], acc[s][1], acc[s][2], acc[s][3]);
                if (b4 == nb4 - 1) {
                    *reinterpret_cast<uint4*>(hrow + size_t(s) * HS + 4) = make_uint4(TG_INFU, TG_INFU, TG_INFU, TG_INFU);
                    *reinterpret_cast<uint4*>(hrow + size_t(s) * HS + 8) = make_uint4(TG_INFU, TG_INFU, TG_INFU, TG_INFU);
                }
            }
        }
    }
    __syncthreads();

    // ---- phase 2: min-plus product with the thresholded cost tables ------------------------------
    const int nGroups = sm.nGroups;
    const int nGQ = (nGroups + 3) >> 2, nAH = (nb4 + 7) >> 3;
    const int dummy = np;  // all-INF row
    unsigned long long bestKey = TG_KEY_NONE;
    for (int wi = warp; wi < nGQ * nAH; wi += nWarps) {
        const int gq = wi / nAH, ah = wi - gq * nAH;
        const int g = gq * 4 + (lane >> 3), t = ah * 8 + (lane & 7);
        if (g >= nGroups || t >= nb4) continue;
        const int k = sm.grpK[g];
        int pr[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) { const int p = sm.grpPair[g][i]; pr[i] = p == 0xffff ? -1 : p; }
        const int a0 = 4 * t;
        uint32_t acc[4][4];
#pragma unroll
        for (int ai = 0; ai < 4; ++ai)
#pragma unroll
            for (int i = 0; i < 4; ++i) acc[ai][i] = TG_INFU;
        const uint32_t* hp[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) hp[i] = Hs + size_t(pr[i] < 0 ? dummy : pr[i]) * HS + a0;

        if (!sm.useGlobalC) {
            const int dm = sm.dmaxTile[k][t];
            const uint32_t* cb = Cs + sm.baseK[k] + a0;
            uint32_t W[4][8];
            if (dm > 0) {
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const uint4 h = *reinterpret_cast<const uint4*>(hp[i]);
                    W[i][4] = h.x; W[i][5] = h.y; W[i][6] = h.z; W[i][7] = h.w;
                }
            }
            for (int q = 0; 4 * q < dm; ++q) {
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    W[i][0] = W[i][4]; W[i][1] = W[i][5]; W[i][2] = W[i][6]; W[i][3] = W[i][7];
                    const uint4 h = *reinterpret_cast<const uint4*>(hp[i] + 4 * q + 4);
                    W[i][4] = h.x; W[i][5] = h.y; W[i][6] = h.z; W[i][7] = h.w;
                }
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int d = 4 * q + 1 + e;
                    uint4 c4 = make_uint4(TG_INFU, TG_INFU, TG_INFU, TG_INFU);
                    if (d <= dm) c4 = *reinterpret_cast<const uint4*>(cb + sm.rowOffS[d]);
                    const uint32_t cv[4] = {c4.x, c4.y, c4.z, c4.w};
#pragma unroll
                    for (int ai = 0; ai < 4; ++ai)
#pragma unroll
                        for (int i = 0; i < 4; ++i) acc[ai][i] = tgAddMin(cv[ai], W[i][ai + e], acc[ai][i]);
                }
            }
        } else {
            // cost tables too large for shared memory: read the reduced table from global (L2)
            const uint32_t* cdk = I.cd + size_t(sm.isl[k]) * I.triG;
            const int dm = min(sm.dmaxK[k], L - 1 - a0);
            for (int d = 1; d <= dm; ++d) {
                uint4 c4 = __ldg(reinterpret_cast<const uint4*>(cdk + tgGOff(L, d) + a0));
                const int amax = L - 1 - d;
                uint32_t cv[4] = {c4.x, c4.y, c4.z, c4.w};
#pragma unroll
                for (int ai = 0; ai < 4; ++ai) {
                    if (a0 + ai > amax || cv[ai] > T) cv[ai] = TG_INFU;
#pragma unroll
                    for (int i = 0; i < 4; ++i) acc[ai][i] = tgAddMin(cv[ai], hp[i][ai + d - 1], acc[ai][i]);
                }
            }
        }
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            if (pr[i] < 0) continue;
            *reinterpret_cast<uint4*>(Gcur + (size_t(first) * nk + pr[i]) * Lp + a0) =
                make_uint4(acc[0][i], acc[1][i], acc[2][i], acc[3][i]);
            if (t == 0 && acc[0][i] < TG_INFU) {
                const uint32_t S = uint32_t(sm.tileMask[pr[i] / nk]) | (1u << k);
                const unsigned long long key = (unsigned long long)acc[0][i] << 32 | (unsigned long long)S << 8 | (unsigned long long)k;
                bestKey = key < bestKey ? key : bestKey;
            }
        }
    }
    if (bestKey != TG_KEY_NONE) atomicMin(&sm.tileKey, bestKey);
    __syncthreads();
    if (tid == 0 && sm.tileKey != TG_KEY_NONE) atomicMin(keys + itemIdx, sm.tileKey);
}

// ---------------------------------------------------------------------------------------------
// Level dispatch: CTA c owns the contiguous tile range [N*c/G, N*(c+1)/G) of level r.
// ---------------------------------------------------------------------------------------------
__device__ void tgProcessLevel(const TgSolveCtx& ctx, TgShared& sm, uint32_t* Cs, uint32_t* Hs, int par, int r,
                               int nItems, int round) {
    const uint32_t* pre = ctx.tilePrefix + (size_t(par) * (TG_MAX_K + 1) + r) * (TG_MAX_ITEMS + 1);
    const TgItem* items = ctx.items + size_t(par) * TG_MAX_ITEMS;
    unsigned long long* keys = ctx.keys + size_t(par) * TG_MAX_ITEMS;
    const uint32_t total = __ldcg(pre + nItems);
    const uint32_t t0 = uint32_t(uint64_t(total) * blockIdx.x / gridDim.x);
    const uint32_t t1 = uint32_t(uint64_t(total) * (blockIdx.x + 1) / gridDim.x);
    if (t0 >= t1) return;
    int lo = 0, hi = nItems - 1;  // last item with pre[item] <= t0
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (__ldcg(pre + mid) <= t0) lo = mid; else hi = mid - 1;
    }
    int it = lo;
    for (uint32_t t = t0; t < t1; ++t) {
        while (t >= __ldcg(pre + it + 1)) ++it;
        const int tileInItem = int(t - __ldcg(pre + it));
        const int id = round * TG_MAX_ITEMS + it;
        if (sm.stagedItem != id) tgStageItem(ctx, sm, Cs, Hs, items + it, id);
        if (r == 0) tgLevel0(ctx, sm, items + it, it, keys);
        else tgTile(ctx, sm, Cs, Hs, items + it, it, keys, r, tileInItem);
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------
// Step 7: plan back-tracker.  One warp per kept-table item: re-derive the per-state argmin
// (lowest b, then lowest j — SURVEY A13) along the optimal path from the stored G levels.
// ---------------------------------------------------------------------------------------------
__device__ void tgBacktrack(const TgSolveCtx& ctx, const TgItem* itp, unsigned long long key) {
    const int lane = threadIdx.x & 31;
    TgInstDev& I = ctx.inst[__ldcg(&itp->inst)];
    const int L = I.L, Lp = I.Lp, K = I.K, Ke = __ldcg(&itp->Ke);
    const uint32_t T = __ldcg(&itp->T);
    tg_result* out = ctx.out + __ldcg(&itp->inst);
    TgItem itv;
    itv.off = __ldcg(&itp->off); itv.bufWords = 0; itv.Ke = uint8_t(Ke);
    uint8_t isl[TG_MAX_K];
#pragma unroll
    for (int e = 0; e < TG_MAX_K; ++e) isl[e] = __ldcg(&itp->isl[e]);
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
            const uint32_t* Gl = ctx.scratch + tgLevelOff(itv, Lp, r - 1);
            const uint32_t* cdk = I.cd + size_t(ko) * I.triG;
            unsigned long long best = TG_KEY_NONE;
            for (int bb = a + 1 + lane; bb <= L - 1; bb += 32) {
                const uint32_t c = cdk[tgGOff(L, bb - a) + a];
                if (c > T) continue;
                uint32_t h = TG_INFU; int hj = 0;
                for (int j = 0; j < Ke; ++j) {
                    if (!(R >> j & 1u)) continue;
                    const uint32_t Rp = R ^ (1u << j);
                    const size_t row = size_t(ctx.rankOf[Rp]) * (Ke - r + 1) + (j - __popc(R & ((1u << j) - 1u)));
                    const uint32_t v = I.x[ko * TG_MAX_K + isl[j]] + __ldcg(Gl + row * Lp + bb);
                    if (v < h) { h = v; hj = j; }
                }
                const uint32_t v = c + h;
                if (v >= TG_INFU) continue;
                const unsigned long long kk = (unsigned long long)v << 32 | (unsigned long long)bb << 8 | (unsigned long long)hj;
                best = kk < best ? kk : best;
            }
            for (int o = 16; o > 0; o >>= 1) {
                const unsigned long long ot = __shfl_xor_sync(0xffffffffu, best, o);
                best = ot < best ? ot : best;
            }
            if (best == TG_KEY_NONE) { bad = true; break; }
            b = int(best >> 8) & 0xffffff;
            const int j = int(best & 0xffu);
            sb[n] = a; si[n] = ko; sp[n] = I.argp[size_t(tgSliceIdx(L, a, b)) * K + ko];
            ++n;
            a = b; k = j; R ^= 1u << j;
            continue;
        }
        sb[n] = a; si[n] = ko; sp[n] = I.argp[size_t(tgSliceIdx(L, a, b)) * K + ko];
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
        if (ctx.mode == 1) { z.bottleneck_us = int32_t(Trep); z.iter_time_us = int64_t(val) + int64_t(I.m - 1) * Trep; }
        else { z.bottleneck_us = int32_t(T); z.iter_time_us = I.incIter; }
        for (int e = 0; e < n; ++e) { z.stage_begin[e] = sb[e]; z.stage_island[e] = si[e]; z.stage_plan[e] = sp[e]; }
        *out = z;
    }
}

// ---------------------------------------------------------------------------------------------
// Scheduler (CTA 0): fold results of the previous round, plan the next one.
//   NEW -> INIT   : DP at T = infinity gives f_inf, the lower bound of the stop rule
//   SEARCH        : multi-section search for the lowest feasible candidate (feasibility is monotone)
//   SWEEP         : ascending candidates while  (f_inf + (m-1)T, idx) < (incumbent iter, its idx)
//   FINAL         : DP at T* keeping every level, followed by the back-track
// The incumbent is the lexicographic minimum of (iter, candidate index) over every DP evaluated,
// which equals the oracle's ascending sweep with strict improvement (lowest T wins ties).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ bool tgMustEval(const TgInstDev& I, int idx, bool full) {
    if (full) return true;
    const int64_t lb = int64_t(I.fInf) + int64_t(I.m - 1) * int64_t(I.cand[idx]);
    return lb < I.incIter || (lb == I.incIter && idx < I.incIdx);
}

__device__ __forceinline__ void tgFoldResult(TgInstDev& I, unsigned long long key, int tidx) {
    if (key == TG_KEY_NONE) return;
    const int64_t it = int64_t(key >> 32) + int64_t(I.m - 1) * int64_t(I.cand[tidx]);
    if (it < I.incIter || (it == I.incIter && tidx < I.incIdx)) { I.incIter = it; I.incIdx = tidx; }
}

__device__ void tgSchedule(const TgSolveCtx& ctx, TgShared& sm, uint32_t* dyn, int round) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int par = round & 1, prv = par ^ 1;
    TgCtrl* ctrl = ctx.ctrl;
    TgItem* items = ctx.items + size_t(par) * TG_MAX_ITEMS;
    const TgItem* itemsPrev = ctx.items + size_t(prv) * TG_MAX_ITEMS;
    unsigned long long* keys = ctx.keys + size_t(par) * TG_MAX_ITEMS;
    const unsigned long long* keysPrev = ctx.keys + size_t(prv) * TG_MAX_ITEMS;
    const bool full = (ctx.flags & TG_SOLVE_FULL_SWEEP) != 0;
    const int nInst = ctx.nInst;
    // planner scratch in dynamic shared memory
    uint32_t* kw = dyn;                                        // [TG_MAX_ITEMS]
    uint8_t* itKe = reinterpret_cast<uint8_t*>(dyn + TG_MAX_ITEMS);  // [TG_MAX_ITEMS]
    uint16_t* itLp = reinterpret_cast<uint16_t*>(dyn + TG_MAX_ITEMS + TG_MAX_ITEMS / 4);  // [TG_MAX_ITEMS]

    if (tid == 0) { sm.iTmp[0] = 0; sm.iTmp[1] = 0; sm.iTmp[2] = 0; sm.iTmp[3] = 0; sm.llTmp[0] = 0; sm.llTmp[1] = 0; sm.stagedItem = -1; }
    __syncthreads();

    // ---- A: fold the previous round ---------------------------------------------------------
    int nActive = 0;
    for (int i = tid; i < nInst; i += TG_NT) {
        TgInstDev& I = ctx.inst[i];
        if (I.itemCnt > 0) {
            const int beg = I.itemBeg, cnt = I.itemCnt;
            if (I.phase == TG_PH_INIT) {
                const unsigned long long key = __ldcg(keysPrev + beg);
                I.nrun += 1;
                if (key == TG_KEY_NONE) {
                    tg_result z;
                    memset(&z, 0, sizeof(z));
                    z.iter_time_us = INT64_MAX;
                    z.n_thresholds_run = uint32_t(I.nrun);
                    ctx.out[i] = z;
                    I.phase = TG_PH_DONE;
                } else {
                    I.fInf = uint32_t(key >> 32);
                    const int n = I.ncand;
                    I.incIdx = n - 1;
                    I.incIter = int64_t(I.fInf) + int64_t(I.m - 1) * int64_t(I.cand[n - 1]);
                    if (full) { I.phase = TG_PH_SWEEP; I.next = 0; }
                    else if (n > 1) { I.phase = TG_PH_SEARCH; I.lo = 0; I.hi = n - 1; }
                    else { I.phase = TG_PH_SWEEP; I.next = n; }  // single candidate: already seeded
                }
            } else if (I.phase == TG_PH_SEARCH) {
                int lo = I.lo, hi = I.hi, prevIdx = -1;
                bool found = false;
                for (int q = 0; q < cnt; ++q) {
                    const int tidx = __ldcg(&itemsPrev[beg + q].tidx);
                    const unsigned long long key = __ldcg(keysPrev + beg + q);
                    tgFoldResult(I, key, tidx);
                    if (!found) {
                        if (key != TG_KEY_NONE) { found = true; hi = tidx; if (prevIdx >= 0) lo = prevIdx + 1; }
                        else prevIdx = tidx;
                    }
                }
                if (!found) lo = prevIdx + 1;
                I.lo = lo; I.hi = hi; I.nrun += cnt;
                if (lo >= hi) { I.phase = TG_PH_SWEEP; I.next = hi + 1; }
            } else if (I.phase == TG_PH_SWEEP) {
                int last = I.next;
                for (int q = 0; q < cnt; ++q) {
                    const int tidx = __ldcg(&itemsPrev[beg + q].tidx);
                    tgFoldResult(I, __ldcg(keysPrev + beg + q), tidx);
                    last = tidx + 1;
                }
                I.next = last; I.nrun += cnt;
            } else if (I.phase == TG_PH_FINAL) {
                I.phase = TG_PH_DONE;  // result written by the back-tracker
            }
            I.itemCnt = 0;
        }
        if (I.phase != TG_PH_DONE) ++nActive;
    }
    if (nActive) atomicAdd(&sm.iTmp[0], nActive);
    __syncthreads();
    nActive = sm.iTmp[0];
    if (nActive == 0) {
        if (tid == 0) { ctrl->done = 1; ctrl->nItems[par] = 0; ctrl->nLevels[par] = 0; }
        return;
    }

    // ---- C: wishes ---------------------------------------------------------------------------
    const int capPerInst = max(1, min(32, TG_MAX_ITEMS / nActive));
    uint32_t carry = 0;
    for (int base = 0; base < nInst; base += TG_NT) {
        const int i = base + tid;
        int cnt = 0, kind = 0, first = 0, probes = 0, span = 0;
        if (i < nInst) {
            TgInstDev& I = ctx.inst[i];
            if (I.phase == TG_PH_NEW || I.phase == TG_PH_INIT) {
                I.phase = ctx.mode == 1 ? TG_PH_FINAL : TG_PH_INIT;
            }
            if (I.phase == TG_PH_SWEEP && !(I.next < I.ncand && tgMustEval(I, I.next, full))) I.phase = TG_PH_FINAL;
            if (I.phase == TG_PH_INIT || I.phase == TG_PH_FINAL) { cnt = 1; kind = I.phase; }
            else if (I.phase == TG_PH_SEARCH || I.phase == TG_PH_SWEEP) {
                // size the wish by the scratch an item needs at its first threshold
                const int tix = I.phase == TG_PH_SEARCH ? I.lo : I.next;
                const uint32_t T = I.cand[tix];
                int Ke = 0;
                for (int k = 0; k < I.K; ++k) Ke += I.cminAll[k] <= T ? 1 : 0;
                uint32_t mx = 1;
                for (int q = 0; q < Ke; ++q) mx = max(mx, tgLevelRows(Ke, q));
                const uint64_t est = 2ull * mx * uint64_t(I.Lp) * uint64_t(nActive);
                uint64_t wsh = ctx.softWords / est;
                if (wsh < 1) wsh = 1;
                if (wsh > uint64_t(capPerInst)) wsh = uint64_t(capPerInst);
                const int wish = int(wsh);
                kind = I.phase;
                if (I.phase == TG_PH_SEARCH) {
                    span = I.hi - I.lo;
                    probes = min(wish, span);
                    cnt = probes; first = I.lo;
                } else {
                    first = I.next;
                    int idx = first;
                    while (cnt < wish && idx < I.ncand && tgMustEval(I, idx, full)) { ++cnt; ++idx; }
                }
            }
        }
        uint32_t tot;
        const uint32_t pos = tgBlockExScan(uint32_t(cnt), sm.warpSums, tot) + carry;
        carry += tot;
        if (i < nInst && cnt > 0) {
            TgInstDev& I = ctx.inst[i];
            if (pos + cnt > TG_MAX_ITEMS) cnt = 0;
            I.itemBeg = int(pos); I.itemCnt = cnt;
            if (cnt > 0) atomicMax(&sm.iTmp[1], int(pos) + cnt);
            for (int q = 0; q < cnt; ++q) {
                TgItem& it = items[pos + q];
                it.inst = i;
                if (kind == TG_PH_INIT) { it.tidx = -1; it.T = TG_TINF; it.flags = 0; }
                else if (kind == TG_PH_FINAL) {
                    if (ctx.mode == 1) { it.tidx = -1; it.T = ctx.dpT; }
                    else { it.tidx = I.incIdx; it.T = I.cand[I.incIdx]; }
                    it.flags = 1;
                } else if (kind == TG_PH_SEARCH) {
                    it.tidx = first + int((int64_t(q + 1) * span) / (probes + 1));
                    it.T = I.cand[it.tidx]; it.flags = 0;
                } else { it.tidx = first + q; it.T = I.cand[it.tidx]; it.flags = 0; }
            }
        }
    }
    __syncthreads();
    const int nIt = sm.iTmp[1];

    // ---- D: per-item geometry ----------------------------------------------------------------
    for (int idx = tid; idx < nIt; idx += TG_NT) {
        TgItem& it = items[idx];
        const TgInstDev& I = ctx.inst[it.inst];
        uint32_t alive = 0; int Ke = 0;
        for (int k = 0; k < I.K; ++k)
            if (I.cminAll[k] <= it.T) { alive |= 1u << k; it.isl[Ke++] = uint8_t(k); }
        for (int e = Ke; e < TG_MAX_K; ++e) it.isl[e] = 0;
        it.alive = uint16_t(alive); it.Ke = uint8_t(Ke);
        uint64_t words = 0;
        if (Ke > 0) {
            if (it.flags & 1) { it.bufWords = 0; words = uint64_t(Ke) * (1ull << (Ke - 1)) * uint64_t(I.Lp); }
            else {
                uint32_t mx = 1;
                for (int q = 0; q < Ke; ++q) mx = max(mx, tgLevelRows(Ke, q));
                it.bufWords = uint64_t(mx) * uint64_t(I.Lp);
                words = 2 * it.bufWords;
            }
        } else it.bufWords = 0;
        kw[idx] = uint32_t((words + 1023) >> 10);
        itKe[idx] = uint8_t(Ke);
        itLp[idx] = uint16_t(I.Lp);
    }
    __syncthreads();

    // ---- E: scratch offsets, hard budget -------------------------------------------------------
    uint32_t carryKw = 0;
    const uint32_t budgetKw = uint32_t(ctx.scratchWords >> 10);
    for (int base = 0; base < nIt; base += TG_NT) {
        const int idx = base + tid;
        const uint32_t v = idx < nIt ? kw[idx] : 0u;
        uint32_t tot;
        const uint32_t pos = tgBlockExScan(v, sm.warpSums, tot) + carryKw;
        carryKw += tot;
        if (idx < nIt) {
            items[idx].off = uint64_t(pos) << 10;
            if (pos + v <= budgetKw) atomicAdd(&sm.iTmp[2], 1);
        }
    }
    __syncthreads();
    const int nFit = sm.iTmp[2];

    // ---- F: trim the instances' item ranges; statistics ------------------------------------------
    for (int i = tid; i < nInst; i += TG_NT) {
        TgInstDev& I = ctx.inst[i];
        if (I.itemCnt > 0) {
            if (I.itemBeg >= nFit) I.itemCnt = 0;
            else I.itemCnt = min(I.itemCnt, nFit - I.itemBeg);
        }
    }
    unsigned long long dense = 0, live = 0;
    int maxKe = 0;
    for (int idx = tid; idx < nFit; idx += TG_NT) {
        keys[idx] = TG_KEY_NONE;
        const TgInstDev& I = ctx.inst[items[idx].inst];
        const int Ke = itKe[idx];
        dense += (unsigned long long)I.NS * I.K << (I.K - 1);
        if (Ke) live += (unsigned long long)I.L * Ke << (Ke - 1);
        maxKe = max(maxKe, Ke);
    }
    if (dense) atomicAdd(&sm.llTmp[0], dense);
    if (live) atomicAdd(&sm.llTmp[1], live);
    if (maxKe) atomicMax(&sm.iTmp[3], maxKe);

    // ---- H: per-level tile prefix sums, one warp per level -----------------------------------------
    if (warp < TG_MAX_K) {
        uint32_t* pre = ctx.tilePrefix + (size_t(par) * (TG_MAX_K + 1) + warp) * (TG_MAX_ITEMS + 1);
        uint32_t run = 0;
        for (int base = 0; base < nFit; base += 32) {
            const int idx = base + lane;
            const uint32_t v = idx < nFit ? tgTiles(ctx, itKe[idx], itLp[idx], warp) : 0u;
            uint32_t inc = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += t;
            }
            if (idx < nFit) pre[idx] = run + inc - v;
            run += __shfl_sync(0xffffffffu, inc, 31);
        }
        if (lane == 0) pre[nFit] = run;
    }
    __syncthreads();
    if (tid == 0) {
        ctrl->nItems[par] = nFit;
        ctrl->nLevels[par] = sm.iTmp[3];
        ctrl->stats.n_dp += uint64_t(nFit);
        ctrl->stats.plans_dense += sm.llTmp[0];
        ctrl->stats.states_live += sm.llTmp[1];
        ctrl->stats.n_rounds += 1;
        if (nFit == 0) { ctrl->errFlag = 1; ctrl->done = 1; }
    }
}

// ---------------------------------------------------------------------------------------------
// The persistent kernel
// ---------------------------------------------------------------------------------------------
extern __shared__ uint4 tgDynSmem[];

__global__ void __launch_bounds__(TG_NT, 1) tgSolveKernel(const TgSolveCtx ctx) {
    __shared__ TgShared sm;
    uint32_t* dyn = reinterpret_cast<uint32_t*>(tgDynSmem);
    uint32_t* Cs = dyn;
    uint32_t* Hs = dyn + ctx.csWords;
    uint32_t epoch = 0;
    TgCtrl* ctrl = ctx.ctrl;
    if (threadIdx.x == 0) sm.stagedItem = -1;
    __syncthreads();
    for (int round = 0;; ++round) {
        const int par = round & 1, prv = par ^ 1;
        // back-track the kept-table items of the previous round (their scratch is still intact)
        if (round > 0) {
            const int nPrev = __ldcg(&ctrl->nItems[prv]);
            const TgItem* itemsPrev = ctx.items + size_t(prv) * TG_MAX_ITEMS;
            const unsigned long long* keysPrev = ctx.keys + size_t(prv) * TG_MAX_ITEMS;
            const int gw = blockIdx.x * (TG_NT >> 5) + (threadIdx.x >> 5), nw = gridDim.x * (TG_NT >> 5);
            // CTA 0 is busy scheduling: give it the back-track work last
            for (int idx = nw - 1 - gw; idx < nPrev; idx += nw)
                if (__ldcg(&itemsPrev[idx].flags) & 1) tgBacktrack(ctx, itemsPrev + idx, __ldcg(keysPrev + idx));
        }
        if (blockIdx.x == 0) tgSchedule(ctx, sm, dyn, round);
        tgGridBarrier(ctrl, epoch);
        if (__ldcg(&ctrl->done)) break;
        const int nItems = __ldcg(&ctrl->nItems[par]), nLevels = __ldcg(&ctrl->nLevels[par]);
        for (int r = 0; r < nLevels; ++r) {
            tgProcessLevel(ctx, sm, Cs, Hs, par, r, nItems, round);
            tgGridBarrier(ctrl, epoch);
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) ctrl->stats.n_barriers = epoch;
}
