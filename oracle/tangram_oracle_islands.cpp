// TEST INFRASTRUCTURE — NOT PART OF THE PRODUCT PATH.
//
// CPU oracle for SURVEY.md §8(f) NEXT-4: GPU island construction (§4.1).  Separate translation unit;
// shares no code with the CUDA library.
//
// Input: nodes n = 0..N-1 with gpus[n] GPUs each, every GPU of node n having compute capacity comp[n],
// memory mem_mb[n] and intra-node interconnect bandwidth intra[n]; inter[n][n'] = network bandwidth from node n to node
// n' (directional: "inter-node bandwidths can be asymmetric"); tolerances eps_c, eps_m, eps_i in permille.
//
// Island definition.  A set I of nodes is an island iff
//   (Eq. 1)  all nodes of I have the same number of GPUs, and for every two nodes  max(c)/min(c) <= 1 + eps_c  and
//            max(m)/min(m) <= 1 + eps_m                      -- integer form:  max * 1000 <= min * (1000 + eps)
//   (Eq. 2)  max(b)/min(b) <= 1 + eps_i  for the intra-node bandwidths
//   (Eq. 3)  for every two different nodes n, n' of I and every node n'' outside I:  inter[n][n'] >= inter[n][n''].
//
// Construction (three steps; reading N4 fixes what the paper leaves open):
//   (1) groups by compute / memory: nodes are partitioned by GPU count; inside a part they are sorted by (comp, id) and cut
//       into maximal runs whose largest compute is within 1 + eps_c of the run's smallest; every run is sorted by
//       (mem, id) and cut the same way with eps_m;
//   (2) every group is sorted by (intra, id) and cut into maximal runs within 1 + eps_i;
//   (3) inside every group, greedy agglomerative clustering on the inter-node bandwidth ("to keep the number of islands
//       low"): start from single nodes; repeatedly take, among all pairs of clusters of the group whose union satisfies
//       Eq. 3, the pair with the largest linkage = the slowest link between the two clusters in either direction
//       (complete linkage), ties to the pair with the lowest (smallest node of A, smallest node of B), A before B; merge;
//       stop when no pair of the group can merge.  A single node is always an island (Eq. 3 is empty for it).
// Islands are numbered by their smallest node.  Per island: GPU count = sum of gpus, capacity = the smallest mem_mb of its
// nodes, and between two islands j != k  bw[j][k] = the slowest link from a node of j to a node of k (the activation of
// a pipeline boundary crosses the slowest pair in the worst case); bw[k][k] = the slowest inter-node link inside k, or
// its intra-node bandwidth when it is a single node.
//
// Pins (tests/test_oracle_islands.py): an independent checker of Eq. 1-3 and of the partition on random clusters; no two
// islands of one step-2 group can still be merged (the greedy stop condition, checked independently); the evaluation
// clusters C1 / C2 / C3 of PAPER.md:278-288 (Tab. 3) give 2 / 2 / 4 islands (up to 4 islands on C3);
// hand-worked three-node cases; eps large and uniform links => one island per GPU count; relabelling the nodes
// permutes the islands.

#include <algorithm>
#include <cstdint>
#include <vector>

extern "C" {

// island_of[N] (out), *K_out, island_gpus[<=N], island_cap_mb[<=N], bw[<=N*N] row-major with row length *K_out.
int orc_islands(int N, const int32_t* gpus, const int32_t* comp, const int32_t* mem_mb, const int32_t* intra,
                const int32_t* inter /* [N][N] */, int eps_c, int eps_m, int eps_i, int32_t* island_of, int32_t* K_out,
                int32_t* island_gpus, int32_t* island_cap_mb, int32_t* bw) {
    auto within = [](int64_t hi, int64_t lo, int eps) { return hi * 1000 <= lo * (1000 + int64_t(eps)); };
    // ---- steps 1 and 2: successive run-cutting on (gpus), comp, mem, intra
    std::vector<std::vector<int>> groups;
    {
        std::vector<int> all(N);
        for (int i = 0; i < N; ++i) all[i] = i;
        groups.push_back(all);
        auto cut = [&](const int32_t* key, int eps, bool exact) {
            std::vector<std::vector<int>> next;
            for (auto& g : groups) {
                std::sort(g.begin(), g.end(), [&](int a, int b) { return key[a] != key[b] ? key[a] < key[b] : a < b; });
                std::vector<int> run;
                for (int n : g) {
                    const bool fits = run.empty() || (exact ? key[n] == key[run[0]] : within(key[n], key[run[0]], eps));
                    if (!fits) { next.push_back(run); run.clear(); }
                    run.push_back(n);
                }
                if (!run.empty()) next.push_back(run);
            }
            groups.swap(next);
        };
        cut(gpus, 0, true);
        cut(comp, eps_c, false);
        cut(mem_mb, eps_m, false);
        cut(intra, eps_i, false);
    }
    // ---- step 3: greedy agglomerative clustering inside every group
    std::vector<std::vector<int>> islands;
    auto link = [&](int a, int b) { return int64_t(inter[size_t(a) * N + b]); };
    for (auto& g : groups) {
        std::vector<std::vector<int>> cl;
        for (int n : g) cl.push_back({n});
        while (true) {
            int bi = -1, bj = -1; int64_t bl = -1;
            for (size_t i = 0; i < cl.size(); ++i)
                for (size_t j = 0; j < cl.size(); ++j) {
                    if (i == j) continue;
                    const int mi = *std::min_element(cl[i].begin(), cl[i].end()), mj = *std::min_element(cl[j].begin(), cl[j].end());
                    if (mi > mj) continue;                                   // ordered pair: A holds the smaller node
                    int64_t lk = INT64_MAX;
                    for (int a : cl[i]) for (int b : cl[j]) lk = std::min(lk, std::min(link(a, b), link(b, a)));
                    // Eq. 3 for the union
                    std::vector<int> u = cl[i];
                    u.insert(u.end(), cl[j].begin(), cl[j].end());
                    std::vector<char> in(N, 0);
                    for (int n : u) in[n] = 1;
                    int64_t inner = INT64_MAX, leaving = -1;
                    for (int a : u) for (int b = 0; b < N; ++b) {
                        if (a == b) continue;
                        if (in[b]) inner = std::min(inner, link(a, b)); else leaving = std::max(leaving, link(a, b));
                    }
                    if (inner < leaving) continue;
                    bool better = lk > bl;
                    if (lk == bl && bi >= 0) {
                        const int ci = *std::min_element(cl[bi].begin(), cl[bi].end()), cj = *std::min_element(cl[bj].begin(), cl[bj].end());
                        better = mi < ci || (mi == ci && mj < cj);
                    }
                    if (better) { bl = lk; bi = int(i); bj = int(j); }
                }
            if (bi < 0) break;
            cl[bi].insert(cl[bi].end(), cl[bj].begin(), cl[bj].end());
            cl.erase(cl.begin() + bj);
        }
        for (auto& c : cl) islands.push_back(c);
    }
    std::sort(islands.begin(), islands.end(), [](const std::vector<int>& a, const std::vector<int>& b) {
        return *std::min_element(a.begin(), a.end()) < *std::min_element(b.begin(), b.end());
    });
    const int K = int(islands.size());
    *K_out = K;
    for (int k = 0; k < K; ++k) {
        int g = 0; int32_t cap = INT32_MAX;
        for (int n : islands[k]) { island_of[n] = k; g += gpus[n]; cap = std::min(cap, mem_mb[n]); }
        island_gpus[k] = g; island_cap_mb[k] = cap;
    }
    for (int j = 0; j < K; ++j)
        for (int k = 0; k < K; ++k) {
            int64_t v = INT64_MAX;
            for (int a : islands[j]) for (int b : islands[k]) if (a != b) v = std::min(v, link(a, b));
            if (v == INT64_MAX) v = intra[islands[j][0]];                    // a single-node island's own "link"
            bw[size_t(j) * K + k] = int32_t(v);
        }
    return 0;
}

}  // extern "C"
