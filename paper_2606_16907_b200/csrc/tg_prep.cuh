// Streaming kernels around the DP: input validation, cost-table loader,
// transfer table (step 2), candidate thresholds (step 3) and the pruning pass (step 0, tg_prune).
#pragma once
#include "tg_common.cuh"

// ---------------------------------------------------------------------------------------------
// small helpers
// ---------------------------------------------------------------------------------------------

// slice index s -> (a, b):  s(a,b) = a(2L-a+1)/2 + (b-a-1)
__device__ __forceinline__ void tgSliceAB(int L, int s, int& a, int& b) {
    const float t = float(2 * L + 1);
    int aa = int((t - sqrtf(fmaxf(t * t - 8.0f * float(s), 0.0f))) * 0.5f);
    aa = max(0, min(aa, L - 1));
    while (aa > 0 && aa * (2 * L - aa + 1) / 2 > s) --aa;
    while (aa + 1 < L && (aa + 1) * (2 * L - aa) / 2 <= s) ++aa;
    a = aa;
    b = aa + 1 + (s - aa * (2 * L - aa + 1) / 2);
}

// exclusive block scan of one value per thread (blockDim.x <= 1024, multiple of 32);
// returns the exclusive prefix and writes the block total to `total`.
__device__ __forceinline__ uint32_t tgBlockExScan(uint32_t v, uint32_t* warpSums /*[33]*/, uint32_t& total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    __syncthreads();  // protect warpSums reuse
    if (lane == 31) warpSums[w] = inc;
    __syncthreads();
    if (w == 0) {
        uint32_t s = lane < nw ? warpSums[lane] : 0u, si = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, si, o);
            if (lane >= o) si += t;
        }
        if (lane < nw) warpSums[lane] = si - s;
        if (lane == 31) warpSums[32] = si;
    }
    __syncthreads();
    total = warpSums[32];
    return warpSums[w] + inc - v;
}

// ---------------------------------------------------------------------------------------------
// validation (tg_instance_create): err[0] |= bit per violated rule
// ---------------------------------------------------------------------------------------------
__global__ void tgValidateKernel(const int32_t* __restrict__ time_us, const int32_t* __restrict__ mem_mb,
                                 const int32_t* __restrict__ gpus, const int32_t* __restrict__ cap,
                                 const int32_t* __restrict__ bw, int K, size_t nEntries, int* err) {
    int bad = 0;
    for (size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x; i < nEntries; i += size_t(gridDim.x) * blockDim.x) {
        const int32_t t = time_us[i], mm = mem_mb[i];
        if (t != TG_INVALID && (t < 0 || t > TG_TIME_MAX)) bad |= 1;
        if (mm < 0) bad |= 2;
    }
    if (blockIdx.x == 0 && threadIdx.x < K * K) {
        const int j = threadIdx.x / K, k = threadIdx.x % K;
        if (j != k && bw[threadIdx.x] <= 0) bad |= 4;
        if (j == 0) {
            if (gpus[k] < 1) bad |= 8;
            if (cap[k] < 0) bad |= 16;
        }
    }
    if (bad) atomicOr(err, bad);
}

// tg_instance_create_batch: the same checks for a whole batch, instance = blockIdx.y
struct TgValidateDesc {
    const int32_t *time_us, *mem_mb, *gpus, *cap, *bw;
    int32_t K;
    unsigned long long nEntries;
};
__global__ void tgValidateBatchKernel(const TgValidateDesc* __restrict__ desc, int* err) {
    const TgValidateDesc d = desc[blockIdx.y];
    int bad = 0;
    for (size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x; i < d.nEntries; i += size_t(gridDim.x) * blockDim.x) {
        const int32_t t = d.time_us[i], mm = d.mem_mb[i];
        if (t != TG_INVALID && (t < 0 || t > TG_TIME_MAX)) bad |= 1;
        if (mm < 0) bad |= 2;
    }
    if (blockIdx.x == 0 && int(threadIdx.x) < d.K * d.K) {
        const int j = threadIdx.x / d.K, k = threadIdx.x % d.K;
        if (j != k && d.bw[threadIdx.x] <= 0) bad |= 4;
        if (j == 0) {
            if (d.gpus[k] < 1) bad |= 8;
            if (d.cap[k] < 0) bad |= 16;
        }
    }
    if (bad) atomicOr(err + blockIdx.y, bad);
}

// tg_instance_create_classes: time/mem[s][k][p] = class table[class_of[s]][k][p]; err bit 32 = class index out of range
__global__ void tgExpandClassesKernel(const int32_t* __restrict__ classOf, const int32_t* __restrict__ ctime,
                                      const int32_t* __restrict__ cmem, int nClasses, int L, int KP, size_t nEntries,
                                      int32_t* __restrict__ time_us, int32_t* __restrict__ mem_mb, int* err) {
    int bad = 0;
    for (size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x; i < nEntries; i += size_t(gridDim.x) * blockDim.x) {
        const size_t s = i / size_t(KP), r = i - s * size_t(KP);
        const int c = classOf[s];
        if (c < 0 || c >= nClasses) { bad = 32; time_us[i] = TG_INVALID; mem_mb[i] = 0; continue; }
        if (r == 0) {   // class map of identical layers: the class depends on the slice length only (bit 64 = it does not)
            int a, b;
            tgSliceAB(L, int(s), a, b);
            if (a > 0 && classOf[b - a - 1] != c) bad |= 64;
        }
        time_us[i] = ctime[size_t(c) * KP + r];
        mem_mb[i] = cmem[size_t(c) * KP + r];
    }
    if (bad) atomicOr(err, bad);
}

// tg_instance_set_stages: 0 <= slow <= time on every valid entry, stage counts in [1, 255] (absent: all ones)
__global__ void tgValidateStagesKernel(const int32_t* __restrict__ time_us, const int32_t* __restrict__ slow, int32_t* __restrict__ q,
                                       bool haveQ, size_t n, int* err) {
    int bad = 0;
    for (size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x; i < n; i += size_t(gridDim.x) * blockDim.x) {
        const int32_t t = time_us[i];
        if (t != TG_INVALID && (slow[i] < 0 || slow[i] > t)) bad = 1;
        if (!haveQ) q[i] = 1;
        else if (q[i] < 1 || q[i] > 255) bad = 1;
    }
    if (bad) atomicOr(err, 1);
}

__global__ void tgValidateNonNegKernel(const int32_t* __restrict__ v, size_t n, int* err) {
    int bad = 0;
    for (size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x; i < n; i += size_t(gridDim.x) * blockDim.x)
        if (v[i] < 0 || v[i] > (1 << 20)) bad = 1;
    if (bad) atomicOr(err, 1);
}

// ---------------------------------------------------------------------------------------------
// Step 1: cost-table loader.  One thread per (slice, island) cell at a time, reduction over the P plans.
//   c = min_p { time : time != INVALID, mem <= cap_k }, ties -> lowest p
// Output goes straight into the diagonal-major layout the DP stages from, plus a flat copy for
// the candidate sort.  HBM-bound stream: 8*P bytes read per cell.
// ---------------------------------------------------------------------------------------------
template <bool VEC4>
__device__ __forceinline__ void tgReduceCell(const int32_t* __restrict__ tp, const int32_t* __restrict__ mp,
                                             int P, int32_t capk, uint32_t& best, int& bp) {
    best = TG_INFU;
    bp = 0xff;
    if (VEC4) {
        const int4* t4 = reinterpret_cast<const int4*>(tp);
        const int4* m4 = reinterpret_cast<const int4*>(mp);
        for (int q = 0; q < (P >> 2); ++q) {
            const int4 t = __ldg(t4 + q), mm = __ldg(m4 + q);
            const int32_t tv[4] = {t.x, t.y, t.z, t.w}, mv[4] = {mm.x, mm.y, mm.z, mm.w};
#pragma unroll
            for (int e = 0; e < 4; ++e)
                if (tv[e] != TG_INVALID && mv[e] <= capk && uint32_t(tv[e]) < best) { best = uint32_t(tv[e]); bp = 4 * q + e; }
        }
    } else {
        for (int p = 0; p < P; ++p) {
            const int32_t t = __ldg(tp + p), mm = __ldg(mp + p);
            if (t != TG_INVALID && mm <= capk && uint32_t(t) < best) { best = uint32_t(t); bp = p; }
        }
    }
}

#define TG_LOAD_U 4   // cells per thread of the loader when the batch fills the GPU (1 otherwise)

// outputs of one cell at depth q: the diagonal-major cost, its plan, the sort key
__device__ __forceinline__ void tgLoadEmit(TgInstDev& I, int L, int K, int nCells, int cell, int a, int b, int k, int q,
                                           uint32_t bq, int bp, uint32_t& prev, uint32_t& myMax) {
    const int d = b - a;
    uint32_t* row = I.cd + (size_t(q - 1) * K + k) * I.triG + tgGOff(L, d);
    row[a] = bq;
    if (b == L) {   // last element of the row: write the INF padding up to a multiple of 4
        const int rl = (L - d + 1 + 3) & ~3;
        for (int p = a + 1; p < rl; ++p) row[p] = TG_INFU;
    }
    I.argp[size_t(q - 1) * nCells + cell] = uint8_t(bp);
    // candidate thresholds: every distinct finite cost of any depth (deeper costs repeat the shallower one
    // until a plan stops fitting, so equal neighbours are dropped here already)
    I.sortbuf[size_t(q - 1) * nCells + cell] = (q == I.nDepth || bq != prev) ? bq : TG_INFU;
    prev = bq;
    if (bq < TG_INFU) myMax = max(myMax, bq);
}

// One CTA per 256 * U consecutive cells of one instance; thread t takes cells t, t + 256, ... of the chunk.
// PV > 0: instances with P = 4 * PV plans and no footprint table issue the 2 * PV * U 16-byte loads of their
// cells first and reduce from registers (the stream is bound by the bytes in flight, not by the arithmetic); any
// other instance of the batch takes the cell-at-a-time path.  The slice index is inverted once per thread
// (tgSliceAB) and advanced incrementally: 256 cells further on are 256 / K slices and 256 % K islands further on.
template <int PV, int U>
__global__ void __launch_bounds__(256, (PV == 1 && U > 1) ? 4 : 1) tgLoadKernel(TgInstDev* __restrict__ insts) {
    constexpr int PVA = PV > 0 ? PV : 1;
    TgInstDev& I = insts[blockIdx.y];
    const int L = I.L, K = I.K, P = I.P;
    const int nCells = I.NS * K;
    const int cellFirst = int(blockIdx.x) * (256 * U) + int(threadIdx.x);
    if (int(blockIdx.x) * (256 * U) >= nCells) return;
    __shared__ uint32_t sMin[TG_MAX_K];
    __shared__ int32_t sCap[TG_MAX_K];
    __shared__ uint32_t sMax;
    const bool fast = PV > 0 && P == 4 * PV && I.actmem_mb == nullptr && I.slow_us == nullptr && I.classOf == nullptr;
    int4 tv[U][PVA], mv[U][PVA];
    if (fast) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int cell = cellFirst + 256 * u;
            if (cell < nCells) {
                const int4* t4 = reinterpret_cast<const int4*>(I.time_us + size_t(cell) * P);
                const int4* m4 = reinterpret_cast<const int4*>(I.mem_mb + size_t(cell) * P);
#pragma unroll
                for (int v = 0; v < PVA; ++v) { tv[u][v] = __ldg(t4 + v); mv[u][v] = __ldg(m4 + v); }
            }
        }
    }
    if (threadIdx.x < TG_MAX_K) {
        sMin[threadIdx.x] = TG_INFU;
        sCap[threadIdx.x] = int(threadIdx.x) < K ? __ldg(I.cap_mb + threadIdx.x) : 0;
    }
    if (threadIdx.x == 0) sMax = 0;
    __syncthreads();
    uint32_t myMax = 0;
    if (cellFirst < nCells) {
        const int s0 = cellFirst / K;
        int k = cellFirst - s0 * K, a, b;
        tgSliceAB(L, s0, a, b);
        const int ds = 256 / K, dk = 256 - ds * K;
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int cell = cellFirst + 256 * u;
            if (cell < nCells) {
                const int32_t capk = sCap[k];
                uint32_t best, prev = TG_INFU;
                if (fast) {
                    uint32_t bq = TG_INFU; int bp = 0xff;
#pragma unroll
                    for (int v = 0; v < PVA; ++v) {
                        const int32_t t4[4] = {tv[u][v].x, tv[u][v].y, tv[u][v].z, tv[u][v].w};
                        const int32_t m4[4] = {mv[u][v].x, mv[u][v].y, mv[u][v].z, mv[u][v].w};
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            if (t4[e] != TG_INVALID && m4[e] <= capk && uint32_t(t4[e]) < bq) { bq = uint32_t(t4[e]); bp = 4 * v + e; }
                    }
                    tgLoadEmit(I, L, K, nCells, cell, a, b, k, 1, bq, bp, prev, myMax);
                    best = bq;
                } else if (I.slow_us != nullptr) {
                    // NEXT-2 (multi-stage partial plans): the cell's cost steps.  The feasible plans are visited in the order of
                    // (slowest internal stage, time, p); a plan opens a step if it lowers the cost or ties it with a lower p.
                    const size_t e = size_t(cell) * P;
                    const int d = b - a;
                    const size_t off = size_t(k) * I.triG + tgGOff(L, d) + a, stride = size_t(K) * I.triG;
                    unsigned long long prevKey = 0;      // keys are biased by +1: 0 = none visited yet
                    uint32_t bestT = TG_INFU;
                    int bestP = 0xff, nsteps = 0;
                    best = TG_INFU;
                    while (true) {
                        unsigned long long next = ~0ull;
                        for (int p = 0; p < P; ++p) {
                            const int32_t t = __ldg(I.time_us + e + p);
                            if (t == TG_INVALID || __ldg(I.mem_mb + e + p) > capk) continue;
                            const unsigned long long key = ((unsigned long long)uint32_t(__ldg(I.slow_us + e + p)) << 34 | (unsigned long long)uint32_t(t) << 8 | (unsigned long long)p) + 1ull;
                            if (key > prevKey && key < next) next = key;
                        }
                        if (next == ~0ull) break;
                        prevKey = next;
                        const unsigned long long kk = next - 1ull;
                        const uint32_t sl = uint32_t(kk >> 34), t = uint32_t(kk >> 8) & 0x3ffffffu;
                        const int p = int(kk & 0xffu);
                        if (t < bestT || (t == bestT && p < bestP)) {
                            bestT = t; bestP = p;
                            I.thr[nsteps * stride + off] = sl;
                            I.cd[nsteps * stride + off] = t;
                            I.argp[size_t(nsteps) * nCells + cell] = uint8_t(p);
                            I.sortbuf[size_t(nsteps) * nCells + cell] = sl;
                            if (nsteps == 0) best = sl;            // the cell becomes admissible at its first step
                            myMax = max(myMax, sl);
                            ++nsteps;
                        }
                    }
                    for (int j = nsteps; j < I.nLayers; ++j) {
                        I.thr[j * stride + off] = TG_INFU;
                        I.cd[j * stride + off] = TG_INFU;
                        I.argp[size_t(j) * nCells + cell] = 0xff;
                        I.sortbuf[size_t(j) * nCells + cell] = TG_INFU;
                    }
                    if (b == L) {   // last element of the row: INF padding up to a multiple of 4, in every layer
                        const int rl = (L - d + 1 + 3) & ~3;
                        for (int j = 0; j < I.nLayers; ++j)
                            for (int pp = a + 1; pp < rl; ++pp) {
                                I.thr[j * stride + off + (pp - a)] = TG_INFU;
                                I.cd[j * stride + off + (pp - a)] = TG_INFU;
                            }
                    }
                } else if (I.classOf != nullptr) {
                    // NEXT-3(a): the cell's plans are those of its slice's signature class -- nClasses * K * P entries are
                    // read (and stay in L2) instead of NS * K * P
                    const size_t e = (size_t(__ldg(I.classOf + cell / K)) * K + k) * P;
                    uint32_t bq; int bp;
                    if ((P & 3) == 0) tgReduceCell<true>(I.ctime + e, I.cmem + e, P, capk, bq, bp);
                    else tgReduceCell<false>(I.ctime + e, I.cmem + e, P, capk, bq, bp);
                    tgLoadEmit(I, L, K, nCells, cell, a, b, k, 1, bq, bp, prev, myMax);
                    if (I.cdT && a == 0) I.cdT[k * (L + 2) + (b - a)] = bq;
                    best = bq;
                } else {
                    const size_t e = size_t(cell) * P;
                    best = TG_INFU;
                    for (int q = I.nDepth; q >= 1; --q) {
                        // depth q: the stage holds q microbatches in flight: feasible iff
                        // mem + q * actmem <= cap.  Without an actmem table there is the one static test.
                        uint32_t bq; int bp;
                        if (I.actmem_mb == nullptr) {
                            if ((P & 3) == 0) tgReduceCell<true>(I.time_us + e, I.mem_mb + e, P, capk, bq, bp);
                            else tgReduceCell<false>(I.time_us + e, I.mem_mb + e, P, capk, bq, bp);
                        } else {
                            bq = TG_INFU; bp = 0xff;
                            for (int p = 0; p < P; ++p) {
                                const int32_t t = __ldg(I.time_us + e + p);
                                const long long need = (long long)__ldg(I.mem_mb + e + p) + (long long)q * __ldg(I.actmem_mb + e + p);
                                if (t != TG_INVALID && need <= (long long)capk && uint32_t(t) < bq) { bq = uint32_t(t); bp = p; }
                            }
                        }
                        tgLoadEmit(I, L, K, nCells, cell, a, b, k, q, bq, bp, prev, myMax);
                        best = bq;   // ends up as the depth-1 cost (the least constrained)
                    }
                }
                if (best < sMin[k]) atomicMin(&sMin[k], best);
                // the thread's next cell: 256 cells = ds slices and dk islands further on
                int adv = ds;
                k += dk;
                if (k >= K) { k -= K; ++adv; }
                int pos = b - a - 1 + adv;
                while (a < L && pos >= L - a) { pos -= L - a; ++a; }
                b = a + 1 + pos;
            }
        }
    }
    myMax = __reduce_max_sync(0xffffffffu, myMax);
    if ((threadIdx.x & 31) == 0 && myMax) atomicMax(&sMax, myMax);
    __syncthreads();
    if (threadIdx.x < K && sMin[threadIdx.x] < TG_INFU) atomicMin(&I.cminAll[threadIdx.x], sMin[threadIdx.x]);
    if (threadIdx.x == 0 && sMax) atomicMax(&I.maxKey, sMax);
}

// Step 1 for batches of plain instances (P = 4 * PV plans, no footprint / stage tables), the HBM-bound stream of the path
// (385 MB at the 1024-instance batch).  A CTA takes TG_LOAD_RG consecutive start rows a0 .. a0+7 of one instance -- a
// contiguous stretch of the raw tables -- reduces its cells from registers (16-byte loads, U cells of a thread in flight)
// and collects the reduced costs in a shared-memory tile [island][diagonal][8 starts]; the tile is then written to the
// diagonal-major tables as 32-byte runs (two 16-byte stores of neighbouring lanes = one full sector).  The cell-order
// kernel above writes one 4-byte word per sector there (12 sectors per store request, profiles/r1c_ncu_cfg5_loader.md).
#define TG_LOAD_RG 8
// CTAs of 128 threads: eight of them share an SM instead of four of 256, so the phases of a CTA that move no data (tile
// initialisation, the barriers, the tail of the cell loop) are covered by more neighbours -- 0.109 -> 0.102 ms on the
// 1024-instance batch (64 threads: 0.148 ms, 96: 0.109, 8 cells a thread in flight: 0.127 at 109 registers)
#ifndef TG_LR_NT
#define TG_LR_NT 128
#endif
template <int PV, int U>
__global__ void __launch_bounds__(TG_LR_NT) tgLoadRowsKernel(TgInstDev* __restrict__ insts) {
    extern __shared__ uint32_t tile[];   // [K][L][TG_LOAD_RG]
    TgInstDev& I = insts[blockIdx.y];
    const int L = I.L, K = I.K;
    const int a0 = int(blockIdx.x) * TG_LOAD_RG;
    if (a0 >= L) return;
    const int a1 = min(L, a0 + TG_LOAD_RG);
    const int nCells = I.NS * K;
    const int cellBeg = tgSliceIdx(L, a0, a0 + 1) * K, cellEnd = a1 < L ? tgSliceIdx(L, a1, a1 + 1) * K : nCells;
    __shared__ uint32_t sMin[TG_MAX_K];
    __shared__ int32_t sCap[TG_MAX_K];
    __shared__ uint32_t sMax;
    const int tid = threadIdx.x;
    for (int w = tid; w < K * L * TG_LOAD_RG; w += TG_LR_NT) tile[w] = TG_INFU;
    if (tid < TG_MAX_K) { sMin[tid] = TG_INFU; sCap[tid] = tid < K ? __ldg(I.cap_mb + tid) : 0; }
    if (tid == 0) sMax = 0;
    __syncthreads();
    uint32_t myMax = 0;
    const int ds = TG_LR_NT / K, dk = TG_LR_NT - ds * K;
    for (int base = cellBeg; base < cellEnd; base += TG_LR_NT * U) {
        int4 tv[U][PV], mv[U][PV];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int cell = base + TG_LR_NT * u + tid;
            if (cell < cellEnd) {
                // (NEXT-3(a): a class instance reads the rows of its slice's signature class)
                const size_t src = I.classOf ? size_t(__ldg(I.classOf + cell / K)) * K + size_t(cell % K) : size_t(cell);
                const int4* t4 = reinterpret_cast<const int4*>((I.classOf ? I.ctime : I.time_us) + src * (4 * PV));
                const int4* m4 = reinterpret_cast<const int4*>((I.classOf ? I.cmem : I.mem_mb) + src * (4 * PV));
#pragma unroll
                for (int v = 0; v < PV; ++v) { tv[u][v] = __ldg(t4 + v); mv[u][v] = __ldg(m4 + v); }
            }
        }
        const int cellFirst = base + tid;
        if (cellFirst < cellEnd) {
            const int s0 = cellFirst / K;
            int k = cellFirst - s0 * K, a, b;
            tgSliceAB(L, s0, a, b);
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int cell = cellFirst + TG_LR_NT * u;
                if (cell < cellEnd) {
                    const int32_t capk = sCap[k];
                    uint32_t bq = TG_INFU; int bp = 0xff;
#pragma unroll
                    for (int v = 0; v < PV; ++v) {
                        const int32_t t4[4] = {tv[u][v].x, tv[u][v].y, tv[u][v].z, tv[u][v].w};
                        const int32_t m4[4] = {mv[u][v].x, mv[u][v].y, mv[u][v].z, mv[u][v].w};
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            if (t4[e] != TG_INVALID && m4[e] <= capk && uint32_t(t4[e]) < bq) { bq = uint32_t(t4[e]); bp = 4 * v + e; }
                    }
                    tile[(k * L + (b - a - 1)) * TG_LOAD_RG + (a - a0)] = bq;
                    if (I.cdT && a == 0) I.cdT[k * (L + 2) + (b - a)] = bq;
                    I.argp[cell] = uint8_t(bp);
                    I.sortbuf[cell] = bq;
                    if (bq < TG_INFU) myMax = max(myMax, bq);
                    if (bq < sMin[k]) atomicMin(&sMin[k], bq);
                    // the thread's next cell: TG_LR_NT cells = ds slices and dk islands further on
                    int adv = ds;
                    k += dk;
                    if (k >= K) { k -= K; ++adv; }
                    int pos = b - a - 1 + adv;
                    while (a < L && pos >= L - a) { pos -= L - a; ++a; }
                    b = a + 1 + pos;
                }
            }
        }
    }
    myMax = __reduce_max_sync(0xffffffffu, myMax);
    if ((tid & 31) == 0 && myMax) atomicMax(&sMax, myMax);
    __syncthreads();
    // tile -> diagonal-major rows: row d of island k holds a = 0 .. L-d, padded with INF to a multiple of 4 words; this
    // CTA owns the starts a0 .. a0+7 of every row that reaches them
    const int nd = L - a0;                                   // diagonals with an entry at start a0
    for (int w = tid; w < K * nd * 2; w += TG_LR_NT) {
        const int q = w & 1, r = w >> 1, k = r / nd, d = 1 + (r - k * nd);
        const int a = a0 + 4 * q, rl = (L - d + 1 + 3) & ~3;  // padded row length
        if (a < rl)
            *reinterpret_cast<uint4*>(I.cd + size_t(k) * I.triG + tgGOff(L, d) + a) =
                *reinterpret_cast<const uint4*>(tile + (k * L + (d - 1)) * TG_LOAD_RG + 4 * q);
    }
    if (tid < K && sMin[tid] < TG_INFU) atomicMin(&I.cminAll[tid], sMin[tid]);
    if (tid == 0 && sMax) atomicMax(&I.maxKey, sMax);
}

// ---------------------------------------------------------------------------------------------
// Steps 2-3 and per-instance DP metadata.  One CTA per instance.
//   x[j][k] = ceil(act_mb*1000 / bw[j][k])
//   sufMin[k][d] = min over d' >= d, a <= L-1-d' of c[a][a+d'][k]  (widest admissible diagonal at T)
//   cand = ascending distinct finite c                            (PAPER.md:250 (1))
// Sort: bitonic network on a power-of-two buffer, in shared memory when it fits, else in place in
// global memory (L2 resident).
// ---------------------------------------------------------------------------------------------
// Stable LSD radix sort of A[0..n) (32-bit keys); B is scratch of the same size.  One CTA of TG_PREP_NT
// threads; hist = 32 warps x 2^DB digits in shared memory.  Keys are either finite (<= maxKey) or TG_INFU:
// they are sorted by  key' = min(key, maxKey + 1), which has nbits = bits(maxKey + 1) significant bits, in
// ceil(nbits / DB) passes of DB = 8 or 9 bits (the paper-shaped tables need 17-19 bits: 2 passes of 9 instead
// of 4 of 8).  Returns the buffer that holds the result.
__device__ uint32_t* tgRadixSort(uint32_t* A, uint32_t* B, int n, uint32_t maxKey, uint32_t* hist, uint32_t* warpSums) {
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5, nW = blockDim.x >> 5;
    const int chunk = (((n + nW - 1) / nW) + 31) & ~31;
    const int beg = min(n, w * chunk), end = min(n, beg + chunk);
    const uint32_t cap = maxKey + 1u;
    const int nbits = 32 - __clz(cap);
    const int DB = (nbits + 8) / 9 < (nbits + 7) / 8 ? 9 : 8;     // 9-bit digits only when they save a pass
    const int nPass = (nbits + DB - 1) / DB, NB = 1 << DB;
    const uint32_t dmask = uint32_t(NB - 1);
    uint32_t* myHist = hist + w * NB;
    uint32_t *src = A, *dst = B;
    for (int pass = 0; pass < nPass; ++pass) {
        const int shift = DB * pass;
        for (int e = tid; e < nW * NB; e += blockDim.x) hist[e] = 0;
        __syncthreads();
        for (int b0 = beg; b0 < end; b0 += 128) {   // four groups of 32 keys, loaded together (one L2 latency, not four)
            uint32_t v4[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) { const int i = b0 + 32 * e + lane; v4[e] = i < end ? __ldcg(src + i) : 0u; }
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int i = b0 + 32 * e + lane;
                const uint32_t d = i < end ? (min(v4[e], cap) >> shift) & dmask : uint32_t(NB + lane);
                const uint32_t peers = __match_any_sync(0xffffffffu, d);
                if (d < uint32_t(NB) && lane == __ffs(peers) - 1) myHist[d] += __popc(peers);
                __syncwarp();
            }
        }
        __syncthreads();
        {   // exclusive scan in (digit major, warp minor) order; each thread owns `per` consecutive entries
            const int per = (nW * NB) / blockDim.x;   // 8 or 16 for 32 warps
            uint32_t loc[16], sum = 0;
#pragma unroll
            for (int q = 0; q < 16; ++q)
                if (q < per) { const int e = tid * per + q; loc[q] = hist[(e % nW) * NB + e / nW]; sum += loc[q]; }
            uint32_t tot;
            uint32_t run = tgBlockExScan(sum, warpSums, tot);
#pragma unroll
            for (int q = 0; q < 16; ++q)
                if (q < per) { const int e = tid * per + q; hist[(e % nW) * NB + e / nW] = run; run += loc[q]; }
        }
        __syncthreads();
        for (int b0 = beg; b0 < end; b0 += 128) {   // groups in index order (stability), loads up front
            uint32_t v4[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) { const int i = b0 + 32 * e + lane; v4[e] = i < end ? __ldcg(src + i) : 0u; }
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int i = b0 + 32 * e + lane;
                const uint32_t v = v4[e];
                const uint32_t d = i < end ? (min(v, cap) >> shift) & dmask : uint32_t(NB + lane);
                const uint32_t peers = __match_any_sync(0xffffffffu, d);
                uint32_t pos = 0;
                if (d < uint32_t(NB)) pos = myHist[d] + __popc(peers & ((1u << lane) - 1u));
                __syncwarp();
                if (d < uint32_t(NB)) {
                    dst[pos] = v;
                    if (lane == __ffs(peers) - 1) myHist[d] += __popc(peers);
                }
                __syncwarp();
            }
        }
        __syncthreads();
        uint32_t* t = src; src = dst; dst = t;
    }
    return src;
}

#define TG_PREP_NT 1024
#define TG_SORT_SMEM_MAX 32768    // words of dynamic shared memory of the prepare kernel (key bitmap of 2^20 bits; radix histograms need half)

__global__ void __launch_bounds__(TG_PREP_NT) tgPrepareKernel(TgInstDev* __restrict__ insts) {
    extern __shared__ uint32_t sbuf[];
    __shared__ uint32_t warpSums[33];
    __shared__ uint32_t sMaxX;
    TgInstDev& I = insts[blockIdx.x];
    const int L = I.L, K = I.K, tid = threadIdx.x;
    if (tid == 0) { sMaxX = 0; I.prepCyc[0] = clock64(); }
    __syncthreads();
    // transfer table (per activation-size class when the instance has per-boundary sizes; I.x = the first class)
    const int nCls = max(I.nAct, 1);
    for (int w = tid; w < K * K * nCls; w += TG_PREP_NT) {
        const int cls = w / (K * K), e = w - cls * K * K, j = e / K, k = e % K;
        uint32_t v = 0;
        if (j != k) {
            const int64_t num = int64_t(I.nAct ? I.actVal[cls] : I.act_mb) * 1000, den = I.bw_gbps[e];
            const int64_t q = (num + den - 1) / den;
            v = q > TG_TIME_MAX ? TG_INFU : uint32_t(q);
        }
        if (cls == 0) I.x[j * TG_MAX_K + k] = v;
        if (I.nAct) I.xAct[cls * (TG_MAX_K * TG_MAX_K) + j * TG_MAX_K + k] = v;
        // transfer bound (NEXT-3(b)): the finite transfer times are candidate thresholds too
        if (I.xbound) {
            const bool fin = j != k && v < TG_INFU;
            I.sortbuf[size_t(I.NS) * K * I.nTables + w] = fin ? v : TG_INFU;
            if (fin) atomicMax(&sMaxX, v);
        }
    }
    // row minima (b <= L-1 only) then suffix minima over the diagonal index
    uint32_t* sm = I.sufMin;
    uint32_t* sma = I.sufMinAll;
    const int stride = L + 2;
    for (int w = tid; w < K * (L + 2); w += TG_PREP_NT) {
        const int k = w / stride, d = w - k * stride;
        uint32_t mn = TG_INFU, mnAll = TG_INFU;
        if (d >= 1 && d <= L) {
            // the row holds a = 0..L-d, padded with INF to a multiple of 4 words and 16-byte aligned: 16-byte loads,
            // four in flight; the last element (b = L) only counts for the all-slices minimum
            // (NEXT-2: a slice is admissible from the threshold of its first cost step on)
            const uint4* row4 = reinterpret_cast<const uint4*>((I.nLayers ? I.thr : I.cd) + size_t(k) * I.triG + tgGOff(L, d));
            const int n4 = (L - d + 4) >> 2, last = L - d;
            for (int q0 = 0; q0 < n4; q0 += 4) {
                uint4 v[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) v[e] = q0 + e < n4 ? __ldcg(row4 + q0 + e) : make_uint4(TG_INFU, TG_INFU, TG_INFU, TG_INFU);
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const uint32_t w[4] = {v[e].x, v[e].y, v[e].z, v[e].w};
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        mnAll = min(mnAll, w[c]);
                        if (4 * (q0 + e) + c != last) mn = min(mn, w[c]);
                    }
                }
            }
        }
        sbuf[w] = mn;                 // (shared memory: the suffix scan below is a chain of dependent accesses)
        sbuf[K * stride + w] = mnAll;
    }
    __syncthreads();
    if (tid < 2 * K) {
        uint32_t* s2 = sbuf + tid * stride;   // rows 0..K-1: b <= L-1 only, rows K..2K-1: every slice
        uint32_t run = TG_INFU;
        for (int d = L + 1; d >= 0; --d) { run = min(run, s2[d]); s2[d] = run; }
    }
    __syncthreads();
    for (int w = tid; w < K * stride; w += TG_PREP_NT) { sm[w] = sbuf[w]; sma[w] = sbuf[K * stride + w]; }
    __syncthreads();
    if (tid == 0) I.prepCyc[1] = clock64();
    // Step 3, candidate thresholds = ascending distinct finite keys.  The keys are bounded by maxKey, which for
    // microsecond stage times is far below the number of bits shared memory holds (2^20): mark every key in a
    // bitmap with shared-memory atomics and read the set bits back in order -- O(n + maxKey/32) instead of a sort.
    // Larger keys: stable LSD radix sort (8- or 9-bit digits, per-warp histograms, ping-pong between two global
    // buffers) followed by a unique pass.
    const int n = I.NS * K * I.nTables + (I.xbound ? K * K * max(I.nAct, 1) : 0);
    const uint32_t maxKey = max(I.maxKey, sMaxX);
    const uint32_t nWords = (maxKey >> 5) + 1u;
    uint32_t base = 0;
    if (nWords <= uint32_t(TG_SORT_SMEM_MAX)) {
        for (uint32_t w = tid; w < nWords; w += TG_PREP_NT) sbuf[w] = 0u;
        __syncthreads();
        for (int i0 = 0; i0 < n; i0 += 4 * TG_PREP_NT) {   // four independent loads a thread
            uint32_t v[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) { const int i = i0 + e * TG_PREP_NT + tid; v[e] = i < n ? __ldcg(I.sortbuf + i) : TG_INFU; }
#pragma unroll
            for (int e = 0; e < 4; ++e) if (v[e] <= maxKey) atomicOr(&sbuf[v[e] >> 5], 1u << (v[e] & 31u));
        }
        __syncthreads();
        if (tid == 0) I.prepCyc[2] = clock64();
        const uint32_t per = (nWords + TG_PREP_NT - 1) / TG_PREP_NT, w0 = uint32_t(tid) * per;
        uint32_t cnt = 0;
        for (uint32_t q = 0; q < per; ++q) cnt += (w0 + q < nWords) ? uint32_t(__popc(sbuf[w0 + q])) : 0u;
        uint32_t tot;
        uint32_t pos = tgBlockExScan(cnt, warpSums, tot);
        for (uint32_t q = 0; q < per && w0 + q < nWords; ++q) {
            uint32_t bits = sbuf[w0 + q];
            while (bits) {
                I.cand[pos++] = ((w0 + q) << 5) + uint32_t(__ffs(bits) - 1);
                bits &= bits - 1u;
            }
        }
        base = tot;
        __syncthreads();   // the bitmap is overwritten below
    } else {
        uint32_t* buf = tgRadixSort(I.sortbuf, I.sortbuf2, n, maxKey, sbuf, warpSums);
        if (tid == 0) I.prepCyc[2] = clock64();
        // unique, finite only
        for (int i0 = 0; i0 < n; i0 += 4 * TG_PREP_NT) {   // four consecutive keys a thread: one block scan per 4096 keys
            const int i = i0 + 4 * tid;
            uint32_t v[5], f[4], cnt = 0;
            v[0] = (i > 0 && i < n) ? __ldcg(buf + i - 1) : 0xffffffffu;   // left neighbour of the thread's first key
#pragma unroll
            for (int e = 0; e < 4; ++e) v[e + 1] = i + e < n ? __ldcg(buf + i + e) : 0xffffffffu;
#pragma unroll
            for (int e = 0; e < 4; ++e) { f[e] = (v[e + 1] < TG_INFU && (i + e == 0 || v[e] != v[e + 1])) ? 1u : 0u; cnt += f[e]; }
            uint32_t tot;
            uint32_t pos = base + tgBlockExScan(cnt, warpSums, tot);
#pragma unroll
            for (int e = 0; e < 4; ++e) if (f[e]) I.cand[pos++] = v[e + 1];
            base += tot;
        }
    }
    if (tid == 0) { I.ncand = int(base); I.prepCyc[3] = clock64(); }
    // (the suffix minima go to shared memory for the search below: it is a chain of dependent reads)
    uint32_t* smaS = sbuf;
    for (int w = tid; w < K * stride; w += TG_PREP_NT) smaS[w] = sma[w];
    __syncthreads();
    // Necessary condition for feasibility at T: the longest admissible slices of the islands must add
    // up to at least L layers.  lbIdx = first candidate that passes (ncand if none): the threshold
    // search starts there.
    if (tid < 32) {
        const int nc = int(base);
        int lo = 0, hi = nc;
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            const uint32_t T = I.cand[mid];
            int len = 0;
            if (tid < K) {
                const uint32_t* sf = smaS + tid * stride;
                int l2 = 0, h2 = L;
                while (l2 < h2) {
                    const int m2 = (l2 + h2 + 1) >> 1;
                    if (sf[m2] <= T) l2 = m2; else h2 = m2 - 1;
                }
                len = l2;
            }
            for (int o = 16; o > 0; o >>= 1) len += __shfl_xor_sync(0xffffffffu, len, o);
            if (len >= L) hi = mid; else lo = mid + 1;
        }
        if (tid == 0) { I.lbIdx = lo; I.prepCyc[4] = clock64(); }
    }
}

// ---------------------------------------------------------------------------------------------
// tg_reduce read-back: diagonal-major cd -> slice-major c[NS][K]
// ---------------------------------------------------------------------------------------------
__global__ void tgExportKernel(const TgInstDev* __restrict__ insts, int32_t* __restrict__ c_out,
                               int32_t* __restrict__ argp_out, int32_t* __restrict__ x_out) {
    const TgInstDev& I = insts[0];
    const int L = I.L, K = I.K, nCells = I.NS * K;
    for (int cell = blockIdx.x * blockDim.x + threadIdx.x; cell < nCells; cell += gridDim.x * blockDim.x) {
        const int s = cell / K, k = cell - s * K;
        int a, b;
        tgSliceAB(L, s, a, b);
        int layer = 0;
        c_out[cell] = int32_t(tgCostAt(I, 0, size_t(k) * I.triG + tgGOff(L, b - a) + a, TG_TINF, &layer));
        const uint8_t p = I.argp[size_t(layer) * nCells + cell];
        argp_out[cell] = p == 0xff ? -1 : int32_t(p);
    }
    if (blockIdx.x == 0 && threadIdx.x < K * K)
        x_out[threadIdx.x] = int32_t(I.x[(threadIdx.x / K) * TG_MAX_K + threadIdx.x % K]);
}

// ---------------------------------------------------------------------------------------------
// Step 0: pruning pass (SURVEY.md §8(c) rules R1-R4)
// ---------------------------------------------------------------------------------------------
// R1 infeasible, R2 dominated inside one (slice, island) cell, optional R4 bottleneck cap.
// One instance of a pruning batch (tg_prune is a batch of one): grid.y = instance, counts[4 * y + rule].
struct TgPruneDesc {
    int32_t* time_us;
    const int32_t* mem_mb;
    const int32_t* actmem_mb;   // nullptr: no footprint
    const int32_t* cap;
    int L, K, P, nCells;
};

// PV > 0: an instance with P = 4 * PV plans is pruned from registers -- the 16-byte loads of the thread's U cells are
// issued first, the rules run on the register copy and a cell whose column changed is stored back as 16-byte words;
// any other instance of the batch takes the entry-by-entry path.  grid = (cells / (TG_PR_NT U), instances).
// ACT = false: no instance of the batch has a footprint table -- the third dominance axis is compiled out (ncu showed the integer
// pipe at 72 % with it).
// CTAs of TG_PR_NT = 128 threads, TG_PR_U = 4 cells of a P = 4 instance per thread (the 1024-instance batch under ncu: 256 x 2:
// 101.6-102.9 us, 256 x 4: 94.5, 256 x 6: 92.7, 256 x 8: 106.6, 128 x 3: 93.0, 128 x 4: 90.2, 128 x 6: 88.7, 128 x 8: 93.3, 64 x 6: 88.0,
// 64 x 8: 99.8): a CTA lives for two dependent memory trips (its descriptor, then its cells) and little else, so what counts
// is the bytes each resident CTA has in flight and how many CTAs an SM holds.
#ifndef TG_PR_NT
#define TG_PR_NT 128
#endif
#ifndef TG_PR_U
#define TG_PR_U 4
#endif
template <int PV, int U, bool ACT>
__global__ void __launch_bounds__(TG_PR_NT) tgPruneCellKernel(const TgPruneDesc* __restrict__ descs, int mode, int64_t threshold,
                                                         unsigned long long* counts) {
    constexpr int PVA = PV > 0 ? PV : 1, PP = 4 * PVA;
    const TgPruneDesc D = descs[blockIdx.y];
    int32_t* const time_us = D.time_us;
    const int32_t* const mem_mb = D.mem_mb;
    const int32_t* const actmem_mb = ACT ? D.actmem_mb : nullptr;
    const int32_t* const cap = D.cap;
    const int nCells = D.nCells, K = D.K, P = D.P;
    counts += 4 * blockIdx.y;
    if (int(blockIdx.x) * (TG_PR_NT * U) >= nCells) return;
    const int cellFirst = blockIdx.x * (TG_PR_NT * U) + threadIdx.x;
    unsigned c1 = 0, c2 = 0, c4 = 0;
    if (PV > 0 && P == PP) {
        int4 tv[U][PVA], mv[U][PVA], av[U][PVA];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int cell = cellFirst + TG_PR_NT * u;
            if (cell < nCells) {
#pragma unroll
                for (int v = 0; v < PVA; ++v) {
                    tv[u][v] = *(reinterpret_cast<const int4*>(time_us + size_t(cell) * PP) + v);
                    mv[u][v] = __ldg(reinterpret_cast<const int4*>(mem_mb + size_t(cell) * PP) + v);
                    av[u][v] = (ACT && actmem_mb) ? __ldg(reinterpret_cast<const int4*>(actmem_mb + size_t(cell) * PP) + v) : make_int4(0, 0, 0, 0);
                }
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int cell = cellFirst + TG_PR_NT * u;
            if (cell < nCells) {
                int32_t t[PP], mm[PP], am[PP];
#pragma unroll
                for (int v = 0; v < PVA; ++v) {
                    t[4 * v] = tv[u][v].x; t[4 * v + 1] = tv[u][v].y; t[4 * v + 2] = tv[u][v].z; t[4 * v + 3] = tv[u][v].w;
                    mm[4 * v] = mv[u][v].x; mm[4 * v + 1] = mv[u][v].y; mm[4 * v + 2] = mv[u][v].z; mm[4 * v + 3] = mv[u][v].w;
                    am[4 * v] = av[u][v].x; am[4 * v + 1] = av[u][v].y; am[4 * v + 2] = av[u][v].z; am[4 * v + 3] = av[u][v].w;
                }
                const int32_t capk = __ldg(cap + cell % K);
                unsigned kill = 0;
#pragma unroll
                for (int p = 0; p < PP; ++p)   // R1
                    if (t[p] != TG_INVALID && (ACT ? int64_t(mm[p]) + am[p] > capk : mm[p] > capk)) { t[p] = TG_INVALID; kill |= 1u << p; ++c1; }
                // R2, decided on the cell as R1 left it, one pass over the unordered pairs p < q: q kills p iff q <= p on
                // every axis and they differ (a tie goes to the lower index, p); p kills q iff p <= q, tie included.  (The
                // ordered form -- le and eq of (q, p) for every q != p -- spent twice the comparisons: the pass is bound by them.)
                unsigned dead = 0, live = 0;
#pragma unroll
                for (int p = 0; p < PP; ++p) {
                    if (t[p] != TG_INVALID) live |= 1u << p;
#pragma unroll
                    for (int q = p + 1; q < PP; ++q) {
                        const bool leqp = t[q] <= t[p] && mm[q] <= mm[p] && (!ACT || am[q] <= am[p]);   // an INVALID t[q] is never <= a live t[p]
                        const bool lepq = t[p] <= t[q] && mm[p] <= mm[q] && (!ACT || am[p] <= am[q]);
                        if (leqp && !lepq) dead |= 1u << p;
                        if (lepq) dead |= 1u << q;
                    }
                }
                dead &= live;
#pragma unroll
                for (int p = 0; p < PP; ++p)
                    if (dead >> p & 1u) { t[p] = TG_INVALID; ++c2; }
                kill |= dead;
                if (mode == TG_PRUNE_BOTTLENECK) {
#pragma unroll
                    for (int p = 0; p < PP; ++p)
                        if (t[p] != TG_INVALID && int64_t(t[p]) > threshold) { t[p] = TG_INVALID; kill |= 1u << p; ++c4; }
                }
#pragma unroll
                for (int v = 0; v < PVA; ++v)
                    if (kill >> (4 * v) & 0xfu)
                        *(reinterpret_cast<int4*>(time_us + size_t(cell) * PP) + v) = make_int4(t[4 * v], t[4 * v + 1], t[4 * v + 2], t[4 * v + 3]);
            }
        }
    } else {
        for (int u = 0; u < U; ++u) {
            const int cell = cellFirst + TG_PR_NT * u;
            if (cell >= nCells) break;
            int32_t* t = time_us + size_t(cell) * P;
            const int32_t* mm = mem_mb + size_t(cell) * P;
            const int32_t* am = actmem_mb ? actmem_mb + size_t(cell) * P : nullptr;
            const int32_t capk = cap[cell % K];
            // R1: with a footprint the shallowest depth (one microbatch in flight) decides "never feasible"
            for (int p = 0; p < P; ++p)
                if (t[p] != TG_INVALID && int64_t(mm[p]) + (am ? am[p] : 0) > capk) { t[p] = TG_INVALID; ++c1; }
            // R2: q kills p iff q <= p on every axis (time, memory and, if present, footprint) and differs, or ties with q < p
            uint32_t dead[8] = {0, 0, 0, 0, 0, 0, 0, 0};
            for (int p = 0; p < P; ++p) {
                const int32_t tp = t[p];
                if (tp == TG_INVALID) continue;
                const int32_t mp = mm[p], ap = am ? am[p] : 0;
                bool dd = false;
                for (int q = 0; q < P && !dd; ++q) {
                    const int32_t tq = t[q];
                    if (q == p || tq == TG_INVALID) continue;
                    const int32_t mq = mm[q], aq = am ? am[q] : 0;
                    const bool le = tq <= tp && mq <= mp && aq <= ap;
                    const bool eq = tq == tp && mq == mp && aq == ap;
                    dd = le && (!eq || q < p);
                }
                if (dd) dead[p >> 5] |= 1u << (p & 31);
            }
            for (int p = 0; p < P; ++p)
                if (dead[p >> 5] >> (p & 31) & 1u) { t[p] = TG_INVALID; ++c2; }
            if (mode == TG_PRUNE_BOTTLENECK)
                for (int p = 0; p < P; ++p)
                    if (t[p] != TG_INVALID && int64_t(t[p]) > threshold) { t[p] = TG_INVALID; ++c4; }
        }
    }
    // warp-aggregate the counters
    for (int o = 16; o > 0; o >>= 1) {
        c1 += __shfl_down_sync(0xffffffffu, c1, o);
        c2 += __shfl_down_sync(0xffffffffu, c2, o);
        c4 += __shfl_down_sync(0xffffffffu, c4, o);
    }
    if ((threadIdx.x & 31) == 0) {
        if (c1) atomicAdd(counts + 0, (unsigned long long)c1);
        if (c2) atomicAdd(counts + 1, (unsigned long long)c2);
        if (c4) atomicAdd(counts + 3, (unsigned long long)c4);
    }
}

// R3 pre-pass: island capacity from profiled atom throughput.  capOut[k] = floor(2^32 / tau_k)
// (0 = exempt), capOut[K] = sum.  One CTA per instance.
__global__ void tgPruneTauKernel(const TgPruneDesc* __restrict__ descs, long long* capOut) {
    const TgPruneDesc D = descs[blockIdx.x];
    const int32_t* const time_us = D.time_us;
    const int L = D.L, K = D.K, P = D.P;
    capOut += (TG_MAX_K + 1) * blockIdx.x;
    __shared__ unsigned long long tau[TG_MAX_K];
    __shared__ int bad[TG_MAX_K];
    if (threadIdx.x < TG_MAX_K) { tau[threadIdx.x] = 0; bad[threadIdx.x] = 0; }
    __syncthreads();
    for (int w = threadIdx.x; w < K * L; w += blockDim.x) {
        const int k = w / L, l = w - k * L;
        const int32_t* t = time_us + (size_t(tgSliceIdx(L, l, l + 1)) * K + k) * P;
        long long best = TG_INF;
        for (int p = 0; p < P; ++p) if (t[p] != TG_INVALID) best = min(best, (long long)t[p]);
        if (best >= TG_INF) atomicOr(&bad[k], 1);
        else atomicAdd(&tau[k], (unsigned long long)best);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        long long tot = 0;
        for (int k = 0; k < K; ++k) {
            long long C = 0;
            if (!bad[k]) { long long tk = (long long)tau[k]; if (tk < 1) tk = 1; C = (1ll << 32) / tk; }
            capOut[k] = C;
            tot += C;
        }
        capOut[K] = tot;
    }
}

// R3 imbalance: kill every plan of a (slice, island) pair whose atom share mismatches the island's
// capacity share by more than theta (permille).
__global__ void __launch_bounds__(256) tgPruneImbalanceKernel(const TgPruneDesc* __restrict__ descs, const long long* __restrict__ capIn,
                                                              int64_t theta, unsigned long long* counts) {
    const TgPruneDesc D = descs[blockIdx.y];
    int32_t* const time_us = D.time_us;
    const int L = D.L, K = D.K, P = D.P, nCells = D.nCells;
    capIn += (TG_MAX_K + 1) * blockIdx.y;
    counts += 4 * blockIdx.y;
    if (int(blockIdx.x) * 256 >= nCells) return;
    const int cell = blockIdx.x * 256 + threadIdx.x;
    unsigned c3 = 0;
    if (cell < nCells) {
        const int s = cell / K, k = cell - s * K;
        const long long Ck = capIn[k], Ct = capIn[K];
        if (Ck != 0) {
            int a, b;
            tgSliceAB(L, s, a, b);
            const long long len = b - a;
            const bool over = len * Ct * 1000 > theta * Ck * L;
            const bool under = len * Ct * theta < 1000ll * Ck * L;
            if (over || under) {
                int32_t* t = time_us + size_t(cell) * P;
                for (int p = 0; p < P; ++p) if (t[p] != TG_INVALID) { t[p] = TG_INVALID; ++c3; }
            }
        }
    }
    for (int o = 16; o > 0; o >>= 1) c3 += __shfl_down_sync(0xffffffffu, c3, o);
    if ((threadIdx.x & 31) == 0 && c3) atomicAdd(counts + 2, (unsigned long long)c3);
}
