// GPU island construction (§4.1) as a front end of the composition search: from
// per-node profiles to the K islands, their GPU counts, capacities and the inter-island bandwidth matrix that
// tg_instance_create takes.  One CTA; the cluster is tiny (tens of nodes) and the result is needed once per cluster, so
// the kernel is written for clarity: the run-cutting of steps 1-2 is sequential (thread 0), the clustering of step 3
// evaluates all cluster pairs of an iteration in parallel and picks the best with one 64-bit atomicMax.
// Definitions and tie-breaks: DESIGN.md reading N4 (the oracle restates them independently).
#pragma once
#include "tg_common.cuh"

#define TG_ISL_NT 256

struct TgIslandsArgs {
    int N;
    const int32_t *gpus, *comp, *mem, *intra, *inter;   // device; inter = [N][N], sender-major
    int epsC, epsM, epsI;                               // permille
    int32_t *islandOf, *K, *islandGpus, *islandCap, *bw;   // device outputs; bw row length = *K
};

__device__ __forceinline__ bool tgWithin(long long hi, long long lo, int eps) { return hi * 1000 <= lo * (1000 + (long long)eps); }

__global__ void __launch_bounds__(TG_ISL_NT) tgIslandsKernel(const TgIslandsArgs A) {
    __shared__ int grp[TG_MAX_NODES], cl[TG_MAX_NODES], order[TG_MAX_NODES], tmp[TG_MAX_NODES];
    __shared__ unsigned long long bestPair;
    __shared__ int nGroups;
    const int N = A.N, tid = threadIdx.x;
    // ---- steps 1-2: successive cuts of every group into runs of (GPU count: equal) / compute / memory / intra-node bandwidth
    if (tid == 0) {
        for (int n = 0; n < N; ++n) grp[n] = 0;
        int ng = 1;
        for (int pass = 0; pass < 4; ++pass) {
            const int32_t* key = pass == 0 ? A.gpus : (pass == 1 ? A.comp : (pass == 2 ? A.mem : A.intra));
            const int eps = pass == 1 ? A.epsC : (pass == 2 ? A.epsM : A.epsI);
            // order = nodes sorted by (group, key, id): insertion sort
            for (int n = 0; n < N; ++n) {
                int p = n;
                while (p > 0) {
                    const int m = order[p - 1];
                    const bool less = grp[n] != grp[m] ? grp[n] < grp[m] : (key[n] != key[m] ? key[n] < key[m] : n < m);
                    if (!less) break;
                    order[p] = m;
                    --p;
                }
                order[p] = n;
            }
            int next = -1, runFirst = -1, prevGrp = -1;
            for (int q = 0; q < N; ++q) {
                const int n = order[q];
                const bool fits = grp[n] == prevGrp && (pass == 0 ? key[n] == key[runFirst] : tgWithin(key[n], key[runFirst], eps));
                if (!fits) { ++next; runFirst = n; prevGrp = grp[n]; }
                tmp[n] = next;
            }
            for (int n = 0; n < N; ++n) grp[n] = tmp[n];
            ng = next + 1;
        }
        nGroups = ng;
        for (int n = 0; n < N; ++n) cl[n] = n;   // cluster label = its smallest node
    }
    __syncthreads();
    // ---- step 3: greedy agglomerative clustering inside every group (all groups advance together: a merge in one group
    // changes neither the linkage nor the validity of a pair of another group -- Eq. 3 looks at nodes outside the UNION,
    // whatever cluster they belong to -- so the order across groups does not matter)
    for (int iter = 0; iter < N; ++iter) {
        if (tid == 0) bestPair = 0ull;
        __syncthreads();
        for (int pr = tid; pr < N * N; pr += TG_ISL_NT) {
            const int i = pr / N, j = pr - i * N;
            if (i >= j || cl[i] != i || cl[j] != j || grp[i] != grp[j]) continue;   // i, j = smallest nodes of two clusters of one group
            long long lk = 0x7fffffffffffffffll, inner = 0x7fffffffffffffffll, leaving = -1;
            for (int a = 0; a < N; ++a) {
                const bool ina = cl[a] == i || cl[a] == j;
                if (!ina) continue;
                for (int b = 0; b < N; ++b) {
                    if (a == b) continue;
                    const long long e = A.inter[a * N + b];
                    const bool inb = cl[b] == i || cl[b] == j;
                    if (inb) {
                        inner = min(inner, e);
                        if (cl[a] != cl[b]) lk = min(lk, e);     // links between the two clusters, both directions
                    } else {
                        leaving = max(leaving, e);
                    }
                }
            }
            if (inner < leaving) continue;                       // Eq. 3 fails for the union
            // largest linkage, then lowest i, then lowest j
            const unsigned long long key = (unsigned long long)(lk + 1) << 16 | (unsigned long long)(255 - i) << 8 | (unsigned long long)(255 - j);
            atomicMax(&bestPair, key);
        }
        __syncthreads();
        const unsigned long long bp = bestPair;
        if (bp == 0ull) break;
        const int i = 255 - int(bp >> 8 & 0xffu), j = 255 - int(bp & 0xffu);
        __syncthreads();
        for (int n = tid; n < N; n += TG_ISL_NT) if (cl[n] == j) cl[n] = i;
        __syncthreads();
    }
    // ---- outputs: islands numbered by their smallest node
    if (tid == 0) {
        int K = 0;
        for (int n = 0; n < N; ++n) if (cl[n] == n) tmp[n] = K++;
        *A.K = K;
        for (int n = 0; n < N; ++n) A.islandOf[n] = tmp[cl[n]];
        for (int k = 0; k < K; ++k) { A.islandGpus[k] = 0; A.islandCap[k] = 0x7fffffff; }
        for (int n = 0; n < N; ++n) {
            const int k = tmp[cl[n]];
            A.islandGpus[k] += A.gpus[n];
            A.islandCap[k] = min(A.islandCap[k], A.mem[n]);
        }
        nGroups = K;
    }
    __syncthreads();
    const int K = nGroups;
    for (int pr = tid; pr < K * K; pr += TG_ISL_NT) {
        const int j = pr / K, k = pr - j * K;
        long long v = 0x7fffffffffffffffll;
        int firstJ = -1;
        for (int a = 0; a < N; ++a) {
            if (A.islandOf[a] != j) continue;
            if (firstJ < 0) firstJ = a;
            for (int b = 0; b < N; ++b)
                if (a != b && A.islandOf[b] == k) v = min(v, (long long)A.inter[a * N + b]);
        }
        if (v == 0x7fffffffffffffffll) v = A.intra[firstJ];       // a single-node island's own "link"
        A.bw[pr] = int32_t(v);
    }
}
