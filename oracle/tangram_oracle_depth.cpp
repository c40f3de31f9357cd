// TEST INFRASTRUCTURE — NOT PART OF THE PRODUCT PATH.
//
// CPU oracle for SURVEY.md §8(f) NEXT-1: depth-aware activation memory under 1F1B
// (PAPER.md:246 "earlier stages hold more in-flight activations", :248-250, :258(i) "request a plan
// until it is no longer feasible", :324).  Separate translation unit: the core oracle
// (tangram_oracle.cpp) and its pins stay untouched.  Shares no code with the CUDA library.
//
// Model (reading N1): a stage followed by r later stages holds q = r + 1 microbatches in
// flight, so intra-slice plan p of (slice, island k) is feasible at depth q iff
//     mem_mb[e] + q * actmem_mb[e] <= cap_mb[k]                                   (int64)
// and the stage's time is  c_q[a][b][k] = min over feasible p of time (ties -> lowest p).
// Everything else is the core definition: plan = stages tiling [0,L) on distinct islands,
// sum = sum c_q + sum x, T = max c_q, iter = sum + (m-1) T, result = argmin of
// (iter, T, mask, k_0, b_0, k_1, b_1, ...).  Stage i of an n-stage plan has q = n - i.
//
// Second variant in the same unit, SURVEY.md §8(f) NEXT-3(b) / reading A2: the transfer counts toward the
// bottleneck ("communication can be the bottleneck"; each boundary transfer is its own pipeline
// slot).  With the flag `xbound` (reading N3b) a plan's bottleneck is
//     T = max( max_i c_i , max_i x[k_i][k_{i+1}] )
// i.e. at threshold T a transfer is admissible iff x <= T, and the candidate thresholds are the distinct
// finite values of c and of the off-diagonal x.  Everything else is unchanged; xbound = 0 and actmem = null
// (treated as zeros) is the core definition.  Pinned like the depth variant: orc_variant_solve ==
// orc_variant_bruteforce on tiny instances, flag off == core oracle, the optimum never improves when the
// flag is switched on, re-scoring from the raw tables.
//
// Pins (tests/test_oracle_depth.py): orc_depth_solve == orc_depth_bruteforce (literal enumeration)
// on thousands of tiny instances; actmem = 0 reproduces the core oracle bit for bit; raising actmem
// never improves the optimum; a plan re-scored from the raw tables with the depth rule reproduces
// (sum, T, iter).
//
// orc_prune_depth (tg_prune with a footprint: 3-way dominance) is pinned in tests/test_oracle_prune_depth.py:
// a set-based restatement of R1/R2 in Python, the literal enumeration (orc_depth_bruteforce) giving the same
// optimum before and after pruning, zero footprint == the core orc_prune, survivors form an antichain, a
// hand-worked cell, idempotence.

#include <algorithm>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>

namespace {

constexpr int64_t INF = int64_t(1) << 30;
constexpr int32_t INVALID = 0x7fffffff;
constexpr int64_t TIME_MAX = int64_t(1) << 25;
constexpr int MAXK = 16;

struct Inst {
    int L, K, P, m;
    const int32_t *time_us, *mem_mb, *actmem_mb, *cap_mb, *bw_gbps;   // actmem_mb may be null (= zeros)
    int act_mb;
    int xbound = 0;   // NEXT-3(b): transfers are bounded by T as well
    const int32_t* act_b = nullptr;   // NEXT-3(b), second half: activation MB crossing boundary b (entries 1..L-1), or null
    int NS() const { return L * (L + 1) / 2; }
};

inline int sidx(int L, int a, int b) { return a * (2 * L - a + 1) / 2 + (b - a - 1); }

struct Reduced {
    std::vector<int64_t> c;     // [K+1][NS][K]: c[q] for depth q = 1..K (index 0 unused)
    std::vector<int32_t> argp;  // same shape, -1 = none
    std::vector<int64_t> x;     // [K][K]
    int NS, K;
    int64_t C(int q, int s, int k) const { return c[(size_t(q) * NS + s) * K + k]; }
    int32_t A(int q, int s, int k) const { return argp[(size_t(q) * NS + s) * K + k]; }
};

Reduced reduce_tables(const Inst& I) {
    Reduced R;
    const int NS = I.NS(), K = I.K, P = I.P;
    R.NS = NS; R.K = K;
    R.c.assign(size_t(K + 1) * NS * K, INF);
    R.argp.assign(size_t(K + 1) * NS * K, -1);
    for (int q = 1; q <= K; ++q)
        for (int s = 0; s < NS; ++s)
            for (int k = 0; k < K; ++k)
                for (int p = 0; p < P; ++p) {
                    const size_t e = (size_t(s) * K + k) * P + p;
                    if (I.time_us[e] == INVALID) continue;
                    const int64_t am = I.actmem_mb ? int64_t(I.actmem_mb[e]) : 0;
                    if (int64_t(I.mem_mb[e]) + int64_t(q) * am > int64_t(I.cap_mb[k])) continue;
                    const size_t o = (size_t(q) * NS + s) * K + k;
                    if (int64_t(I.time_us[e]) < R.c[o]) { R.c[o] = I.time_us[e]; R.argp[o] = p; }   // strict: lowest p
                }
    R.x.assign(size_t(K) * K, 0);
    for (int j = 0; j < K; ++j)
        for (int k = 0; k < K; ++k) {
            if (j == k) continue;
            const int64_t num = int64_t(I.act_mb) * 1000, den = I.bw_gbps[j * K + k];
            int64_t v = (num + den - 1) / den;
            if (v > TIME_MAX) v = INF;
            R.x[size_t(j) * K + k] = v;
        }
    return R;
}

// Transfer time across boundary b from the stage on island j to the stage on island k.  With per-boundary activation sizes
// (PAPER.md:240 (1) "only transferring stage inputs and outputs": what crosses a boundary is the output of the layer in
// front of it, whose size may differ from layer to layer, e.g. between attention and MoE blocks) it is
//     x_b[j][k] = ceil(act_b[b] * 1000 / bw[j][k])  microseconds,  unusable (INF) above TIME_MAX,
// else the one table of the core path.
inline int64_t xfer(const Inst& I, const Reduced& R, int b, int j, int k) {
    if (!I.act_b) return R.x[size_t(j) * I.K + k];
    if (j == k) return 0;
    const int64_t num = int64_t(I.act_b[b]) * 1000, den = I.bw_gbps[j * I.K + k];
    const int64_t v = (num + den - 1) / den;
    return v > TIME_MAX ? INF : v;
}

std::vector<int64_t> candidates(const Reduced& R, bool xbound) {
    std::vector<int64_t> v;
    for (int64_t c : R.c) if (c < INF) v.push_back(c);
    if (xbound)
        for (int j = 0; j < R.K; ++j)
            for (int k = 0; k < R.K; ++k)
                if (j != k && R.x[size_t(j) * R.K + k] < INF) v.push_back(R.x[size_t(j) * R.K + k]);
    std::sort(v.begin(), v.end());
    v.erase(std::unique(v.begin(), v.end()), v.end());
    return v;
}

// the same with per-boundary activation sizes: under the transfer bound every boundary's finite transfer times are candidates
std::vector<int64_t> candidates(const Inst& I, const Reduced& R) {
    if (!I.act_b || !I.xbound) return candidates(R, I.xbound != 0);
    std::vector<int64_t> v;
    for (int64_t c : R.c) if (c < INF) v.push_back(c);
    for (int b = 1; b < I.L; ++b)
        for (int j = 0; j < I.K; ++j)
            for (int k = 0; k < I.K; ++k)
                if (j != k && xfer(I, R, b, j, k) < INF) v.push_back(xfer(I, R, b, j, k));
    std::sort(v.begin(), v.end());
    v.erase(std::unique(v.begin(), v.end()), v.end());
    return v;
}

inline int64_t sat(int64_t v) { return v >= INF ? INF : v; }

struct DP {
    int L, K;
    std::vector<int32_t> g, h;
    std::vector<uint8_t> gb, hj;
    size_t at(int a, uint32_t S, int k) const { return (size_t(S) * K + k) * (L + 1) + a; }
};
struct Top { int64_t best; uint32_t S; int k; };

// The core recurrence with one change: the first stage of a suffix that uses the islands S has
// depth q = popcount(S) and takes its cost from c_q.
Top run_dp(const Inst& I, const Reduced& R, int64_t T, DP& D, bool keep) {
    const int L = I.L, K = I.K;
    const uint32_t NM = 1u << K;
    D.L = L; D.K = K;
    D.g.assign(size_t(NM) * K * (L + 1), int32_t(INF));
    D.h.assign(size_t(NM) * K * (L + 1), int32_t(INF));
    if (keep) { D.gb.assign(D.g.size(), 0); D.hj.assign(D.g.size(), 0); }
    for (int d = 1; d <= K; ++d) {
        if (d >= 2)
            for (uint32_t Rm = 1; Rm < NM; ++Rm) {
                if (__builtin_popcount(Rm) != d - 1) continue;
                for (int k = 0; k < K; ++k) {
                    if (Rm >> k & 1) continue;
                    for (int b = 1; b < L; ++b) {
                        int64_t best = INF; int bj = 0;
                        for (int j = 0; j < K; ++j) {
                            if (!(Rm >> j & 1)) continue;
                            if (I.xbound && xfer(I, R, b, k, j) > T) continue;   // NEXT-3(b): the transfer is a pipeline slot
                            const int64_t v = sat(xfer(I, R, b, k, j) + D.g[D.at(b, Rm, j)]);
                            if (v < best) { best = v; bj = j; }
                        }
                        D.h[D.at(b, Rm, k)] = int32_t(best);
                        if (keep) D.hj[D.at(b, Rm, k)] = uint8_t(bj);
                    }
                }
            }
        for (uint32_t S = 1; S < NM; ++S) {
            if (__builtin_popcount(S) != d) continue;
            for (int k = 0; k < K; ++k) {
                if (!(S >> k & 1)) continue;
                const uint32_t Rm = S ^ (1u << k);
                for (int a = L - 1; a >= 0; --a) {
                    int64_t best = INF; int bb = 0;
                    for (int b = a + 1; b <= L; ++b) {
                        const int64_t cv = R.C(d, sidx(L, a, b), k);      // depth q = d = popcount(S)
                        if (cv >= INF || cv > T) continue;
                        int64_t cand;
                        if (b == L) cand = (Rm == 0) ? cv : INF;
                        else cand = (Rm == 0) ? INF : sat(cv + D.h[D.at(b, Rm, k)]);
                        if (cand < best) { best = cand; bb = b; }
                    }
                    D.g[D.at(a, S, k)] = int32_t(best);
                    if (keep) D.gb[D.at(a, S, k)] = uint8_t(bb);
                }
            }
        }
    }
    Top t{INF, 0, 0};
    for (uint32_t S = 1; S < NM; ++S)
        for (int k = 0; k < K; ++k)
            if ((S >> k & 1) && D.g[D.at(0, S, k)] < t.best) t = Top{D.g[D.at(0, S, k)], S, k};
    return t;
}

}  // namespace

extern "C" {

struct orc_result {   // same layout as the core oracle's
    int64_t iter_time_us, sum_us, bottleneck_us;
    int32_t n_stages;
    uint32_t island_mask;
    int32_t n_dp_run, n_candidates;
    int32_t stage_begin[MAXK], stage_island[MAXK], stage_plan[MAXK];
};

static void set_infeasible(orc_result* o) { std::memset(o, 0, sizeof(*o)); o->iter_time_us = INT64_MAX; }

// Full ascending sweep with the exact stop rule f_inf + (m-1)T >= incumbent, then a
// choice-keeping run at T* and the back-track.
int orc_variant_solve(int L, int K, int P, int m, const int32_t* time_us, const int32_t* mem_mb, const int32_t* actmem_mb,
                      const int32_t* cap_mb, const int32_t* bw_gbps, int act_mb, int xbound, orc_result* out) {
    Inst I{L, K, P, m, time_us, mem_mb, actmem_mb, cap_mb, bw_gbps, act_mb, xbound};
    Reduced R = reduce_tables(I);
    std::vector<int64_t> cand = candidates(R, xbound != 0);
    set_infeasible(out);
    out->n_candidates = int(cand.size());
    DP D0;
    const Top tinf = run_dp(I, R, INF, D0, false);
    if (tinf.best >= INF) return 0;
    bool have = false; int64_t best_iter = 0, best_T = 0; int n_dp = 0;
    for (int64_t T : cand) {
        if (have && tinf.best + int64_t(m - 1) * T >= best_iter) break;
        DP D; ++n_dp;
        const Top t = run_dp(I, R, T, D, false);
        if (t.best >= INF) continue;
        const int64_t it = t.best + int64_t(m - 1) * T;
        if (!have || it < best_iter) { have = true; best_iter = it; best_T = T; }
    }
    DP D;
    const Top t = run_dp(I, R, best_T, D, true);
    out->iter_time_us = best_iter; out->sum_us = t.best; out->bottleneck_us = best_T;
    out->island_mask = t.S; out->n_dp_run = n_dp;
    int a = 0, k = t.k, n = 0; uint32_t S = t.S;
    while (true) {
        const int b = D.gb[D.at(a, S, k)];
        out->stage_begin[n] = a; out->stage_island[n] = k;
        out->stage_plan[n] = R.A(__builtin_popcount(S), sidx(L, a, b), k);
        ++n;
        if (b == L) break;
        const uint32_t Rm = S ^ (1u << k);
        const int j = D.hj[D.at(b, Rm, k)];
        a = b; S = Rm; k = j;
    }
    out->n_stages = n;
    return 0;
}

// The same search with the schedule of the core oracle's orc_solve, for the K = 16 configs whose plain ascending sweep
// from the lowest candidate would take hours: bisection for the lowest feasible candidate (feasibility is monotone in
// T: every plan admissible at T stays admissible at T' > T, also with the footprint and the transfer bound, which only
// restrict the set of plans per T), then the ascending sweep with the stop rule A7, evaluated in blocks of n_threads
// independent DP(T) calls that are folded in ascending order with the sequential rules.  The arithmetic (reduce_tables,
// candidates, run_dp, back-track) is that of orc_variant_solve; tests/test_oracle_depth.py pins the two against each
// other (value, plan and the number of candidates) and both against the literal enumeration.
int orc_variant_solve_mt(int L, int K, int P, int m, const int32_t* time_us, const int32_t* mem_mb, const int32_t* actmem_mb,
                         const int32_t* cap_mb, const int32_t* bw_gbps, int act_mb, int xbound, int n_threads, orc_result* out) {
    Inst I{L, K, P, m, time_us, mem_mb, actmem_mb, cap_mb, bw_gbps, act_mb, xbound};
    Reduced R = reduce_tables(I);
    std::vector<int64_t> cand = candidates(R, xbound != 0);
    set_infeasible(out);
    out->n_candidates = int(cand.size());
    DP D0;
    const Top tinf = run_dp(I, R, INF, D0, false);
    if (tinf.best >= INF) return 0;
    const int n = int(cand.size());
    if (n_threads < 1) n_threads = 1;
    int n_dp = 0;
    int l = 0, r = n - 1;                    // cand[n-1] is feasible because f_inf is finite
    while (l < r) {
        const int mid = (l + r) / 2;
        DP D; ++n_dp;
        if (run_dp(I, R, cand[mid], D, false).best < INF) r = mid; else l = mid + 1;
    }
    bool have = false; int64_t best_iter = 0, best_T = 0;
    std::vector<Top> res;
    for (int i0 = l; i0 < n; i0 += n_threads) {
        const int cnt = std::min(n_threads, n - i0);
        if (have && tinf.best + int64_t(m - 1) * cand[i0] >= best_iter) break;            // A7
        res.assign(cnt, Top{INF, 0, 0});
        std::vector<std::thread> th;
        for (int t = 0; t < cnt; ++t)
            th.emplace_back([&, t] { DP D; res[t] = run_dp(I, R, cand[i0 + t], D, false); });
        for (auto& x : th) x.join();
        bool stop = false;
        for (int t = 0; t < cnt; ++t) {
            const int64_t T = cand[i0 + t];
            if (have && tinf.best + int64_t(m - 1) * T >= best_iter) { stop = true; break; }
            ++n_dp;
            if (res[t].best >= INF) continue;
            const int64_t it = res[t].best + int64_t(m - 1) * T;
            if (!have || it < best_iter) { have = true; best_iter = it; best_T = T; }    // ties keep the lower T
        }
        if (stop) break;
    }
    DP D;
    const Top t = run_dp(I, R, best_T, D, true);
    out->iter_time_us = best_iter; out->sum_us = t.best; out->bottleneck_us = best_T;
    out->island_mask = t.S; out->n_dp_run = n_dp;
    int a = 0, k = t.k, ns = 0; uint32_t S = t.S;
    while (true) {
        const int b = D.gb[D.at(a, S, k)];
        out->stage_begin[ns] = a; out->stage_island[ns] = k;
        out->stage_plan[ns] = R.A(__builtin_popcount(S), sidx(L, a, b), k);
        ++ns;
        if (b == L) break;
        const uint32_t Rm = S ^ (1u << k);
        const int j = D.hj[D.at(b, Rm, k)];
        a = b; S = Rm; k = j;
    }
    out->n_stages = ns;
    return 0;
}

// Per-boundary activation sizes (second half; PAPER.md:240 (1), :350): act_b[b] MB cross boundary
// b (1 <= b <= L-1; entries 0 and L are ignored).  Same search as orc_variant_solve_mt / literal enumeration as
// orc_variant_bruteforce with the transfer of a boundary taken from xfer().  act_b == null is the scalar act_mb.
int orc_variant_solve_b(int L, int K, int P, int m, const int32_t* time_us, const int32_t* mem_mb, const int32_t* actmem_mb,
                        const int32_t* cap_mb, const int32_t* bw_gbps, int act_mb, const int32_t* act_b, int xbound, orc_result* out) {
    Inst I{L, K, P, m, time_us, mem_mb, actmem_mb, cap_mb, bw_gbps, act_mb, xbound};
    I.act_b = act_b;
    Reduced R = reduce_tables(I);
    std::vector<int64_t> cand = candidates(I, R);
    set_infeasible(out);
    out->n_candidates = int(cand.size());
    DP D0;
    const Top tinf = run_dp(I, R, INF, D0, false);
    if (tinf.best >= INF) return 0;
    bool have = false; int64_t best_iter = 0, best_T = 0; int n_dp = 0;
    for (int64_t T : cand) {
        if (have && tinf.best + int64_t(m - 1) * T >= best_iter) break;
        DP D; ++n_dp;
        const Top t = run_dp(I, R, T, D, false);
        if (t.best >= INF) continue;
        const int64_t it = t.best + int64_t(m - 1) * T;
        if (!have || it < best_iter) { have = true; best_iter = it; best_T = T; }
    }
    DP D;
    const Top t = run_dp(I, R, best_T, D, true);
    out->iter_time_us = best_iter; out->sum_us = t.best; out->bottleneck_us = best_T;
    out->island_mask = t.S; out->n_dp_run = n_dp;
    int a = 0, k = t.k, n = 0; uint32_t S = t.S;
    while (true) {
        const int b = D.gb[D.at(a, S, k)];
        out->stage_begin[n] = a; out->stage_island[n] = k;
        out->stage_plan[n] = R.A(__builtin_popcount(S), sidx(L, a, b), k);
        ++n;
        if (b == L) break;
        const uint32_t Rm = S ^ (1u << k);
        const int j = D.hj[D.at(b, Rm, k)];
        a = b; S = Rm; k = j;
    }
    out->n_stages = n;
    return 0;
}

int orc_depth_solve(int L, int K, int P, int m, const int32_t* time_us, const int32_t* mem_mb, const int32_t* actmem_mb,
                    const int32_t* cap_mb, const int32_t* bw_gbps, int act_mb, orc_result* out) {
    return orc_variant_solve(L, K, P, m, time_us, mem_mb, actmem_mb, cap_mb, bw_gbps, act_mb, 0, out);
}

// Literal enumeration: every cut set and every ordered choice of distinct islands; the depth of
// stage i is known once the plan is complete (q = n - i).
namespace {
struct BF {
    const Inst* I; const Reduced* R;
    std::vector<int64_t> bestkey; bool have = false;
    std::vector<int> ks, bs;
    int64_t n_plans = 0;
    void leaf() {
        const int L = I->L, n = int(ks.size());
        int64_t sum = 0, T = 0; uint32_t mask = 0;
        int a = 0;
        for (int i = 0; i < n; ++i) {
            const int64_t cv = R->C(n - i, sidx(L, a, bs[i]), ks[i]);
            if (cv >= INF) return;
            sum += cv; T = std::max(T, cv); mask |= 1u << ks[i];
            if (i + 1 < n) {
                const int64_t xs = xfer(*I, *R, bs[i], ks[i], ks[i + 1]);
                if (xs >= INF) return;
                sum += xs;
                if (I->xbound) T = std::max(T, xs);
            }
            a = bs[i];
        }
        ++n_plans;
        std::vector<int64_t> key{sum + int64_t(I->m - 1) * T, T, int64_t(mask)};
        for (int i = 0; i < n; ++i) { key.push_back(ks[i]); key.push_back(bs[i]); }
        if (!have || key < bestkey) { have = true; bestkey = key; }
    }
    void rec(int a, uint32_t used) {
        if (a == I->L) { leaf(); return; }
        for (int k = 0; k < I->K; ++k) {
            if (used >> k & 1) continue;
            for (int b = a + 1; b <= I->L; ++b) {
                ks.push_back(k); bs.push_back(b);
                rec(b, used | (1u << k));
                ks.pop_back(); bs.pop_back();
            }
        }
    }
};
}  // namespace

int orc_variant_bruteforce(int L, int K, int P, int m, const int32_t* time_us, const int32_t* mem_mb, const int32_t* actmem_mb,
                           const int32_t* cap_mb, const int32_t* bw_gbps, int act_mb, int xbound, orc_result* out) {
    Inst I{L, K, P, m, time_us, mem_mb, actmem_mb, cap_mb, bw_gbps, act_mb, xbound};
    Reduced R = reduce_tables(I);
    BF bf; bf.I = &I; bf.R = &R;
    bf.rec(0, 0);
    set_infeasible(out);
    if (!bf.have) return 0;
    out->iter_time_us = bf.bestkey[0]; out->bottleneck_us = bf.bestkey[1];
    out->island_mask = uint32_t(bf.bestkey[2]);
    out->sum_us = bf.bestkey[0] - int64_t(m - 1) * bf.bestkey[1];
    const int n = int(bf.bestkey.size() - 3) / 2;
    out->n_stages = n;
    int a = 0;
    for (int i = 0; i < n; ++i) {
        const int k = int(bf.bestkey[3 + 2 * i]), b = int(bf.bestkey[4 + 2 * i]);
        out->stage_begin[i] = a; out->stage_island[i] = k;
        out->stage_plan[i] = R.A(n - i, sidx(L, a, b), k);
        a = b;
    }
    return 0;
}

int orc_variant_bruteforce_b(int L, int K, int P, int m, const int32_t* time_us, const int32_t* mem_mb, const int32_t* actmem_mb,
                             const int32_t* cap_mb, const int32_t* bw_gbps, int act_mb, const int32_t* act_b, int xbound, orc_result* out) {
    Inst I{L, K, P, m, time_us, mem_mb, actmem_mb, cap_mb, bw_gbps, act_mb, xbound};
    I.act_b = act_b;
    Reduced R = reduce_tables(I);
    BF bf; bf.I = &I; bf.R = &R;
    bf.rec(0, 0);
    set_infeasible(out);
    if (!bf.have) return 0;
    out->iter_time_us = bf.bestkey[0]; out->bottleneck_us = bf.bestkey[1];
    out->island_mask = uint32_t(bf.bestkey[2]);
    out->sum_us = bf.bestkey[0] - int64_t(m - 1) * bf.bestkey[1];
    const int n = int(bf.bestkey.size() - 3) / 2;
    out->n_stages = n;
    int a = 0;
    for (int i = 0; i < n; ++i) {
        const int k = int(bf.bestkey[3 + 2 * i]), b = int(bf.bestkey[4 + 2 * i]);
        out->stage_begin[i] = a; out->stage_island[i] = k;
        out->stage_plan[i] = R.A(n - i, sidx(L, a, b), k);
        a = b;
    }
    return 0;
}

int orc_depth_bruteforce(int L, int K, int P, int m, const int32_t* time_us, const int32_t* mem_mb, const int32_t* actmem_mb,
                         const int32_t* cap_mb, const int32_t* bw_gbps, int act_mb, orc_result* out) {
    return orc_variant_bruteforce(L, K, P, m, time_us, mem_mb, actmem_mb, cap_mb, bw_gbps, act_mb, 0, out);
}

// tg_prune oracle for instances WITH a footprint table (SURVEY.md §8(f) NEXT-1 "R2 dominance becomes 3-way";
// DESIGN.md reading N1-prune).  Rules, on the entry e = (slice, island k, plan p):
//   R1  never feasible: the shallowest depth is q = 1, so  mem + 1*actmem > cap  kills;
//   R2  dominated inside its (slice, island) cell on (time, mem, actmem): q kills p iff  tq <= tp, mq <= mp,
//       aq <= ap  with one of them strict, or all three equal and q < p.  Then mq + d*aq <= mp + d*ap at every
//       depth d >= 1, so q is feasible wherever p is and no slower (PAPER.md:43, :360, :258(i));
//   R3 (mode 1, theta per mille) and R4 (mode 2, cap in us) look at the times only and are the core rules.
// R2 is decided on the cell as R1 left it (dominance is a strict partial order plus the index tie-break, so
// every dominated entry has a surviving dominator).  time_us modified in place, counts[4] as in orc_prune.
int orc_prune_depth(int L, int K, int P, int32_t* time_us, const int32_t* mem_mb, const int32_t* actmem_mb,
                    const int32_t* cap_mb, int mode, int64_t threshold, int64_t* counts) {
    const int NS = L * (L + 1) / 2;
    counts[0] = counts[1] = counts[2] = counts[3] = 0;
    auto E = [&](int s, int k, int p) { return (size_t(s) * K + k) * P + p; };
    for (int s = 0; s < NS; ++s) for (int k = 0; k < K; ++k) for (int p = 0; p < P; ++p) {
        const size_t e = E(s, k, p);
        if (time_us[e] != INVALID && int64_t(mem_mb[e]) + int64_t(actmem_mb[e]) > int64_t(cap_mb[k])) { time_us[e] = INVALID; ++counts[0]; }
    }
    for (int s = 0; s < NS; ++s) for (int k = 0; k < K; ++k) {
        std::vector<char> dead(P, 0);
        for (int p = 0; p < P; ++p) {
            const size_t ep = E(s, k, p);
            if (time_us[ep] == INVALID) continue;
            for (int q = 0; q < P; ++q) {
                const size_t eq = E(s, k, q);
                if (q == p || time_us[eq] == INVALID) continue;
                const bool le = time_us[eq] <= time_us[ep] && mem_mb[eq] <= mem_mb[ep] && actmem_mb[eq] <= actmem_mb[ep];
                const bool eqv = time_us[eq] == time_us[ep] && mem_mb[eq] == mem_mb[ep] && actmem_mb[eq] == actmem_mb[ep];
                if (le && (!eqv || q < p)) dead[p] = 1;
            }
        }
        for (int p = 0; p < P; ++p) if (dead[p]) { time_us[E(s, k, p)] = INVALID; ++counts[1]; }
    }
    if (mode == 1) {
        // R3: island capacity share from the profiled atom throughput, slice demand = its length
        std::vector<int64_t> C(K, 0); int64_t Ct = 0;
        for (int k = 0; k < K; ++k) {
            int64_t tau = 0; bool ok = true;
            for (int l = 0; l < L && ok; ++l) {
                int64_t best = INF;
                for (int p = 0; p < P; ++p) { const int32_t t = time_us[E(sidx(L, l, l + 1), k, p)]; if (t != INVALID) best = std::min<int64_t>(best, t); }
                if (best >= INF) ok = false; else tau += best;
            }
            if (ok) { C[k] = (int64_t(1) << 32) / std::max<int64_t>(tau, 1); Ct += C[k]; }
        }
        for (int a = 0; a < L; ++a) for (int b = a + 1; b <= L; ++b) for (int k = 0; k < K; ++k) {
            if (C[k] == 0) continue;
            const int64_t len = b - a;
            const bool over = len * Ct * 1000 > threshold * C[k] * L;
            const bool under = len * Ct * threshold < int64_t(1000) * C[k] * L;
            if (!(over || under)) continue;
            for (int p = 0; p < P; ++p) { const size_t e = E(sidx(L, a, b), k, p); if (time_us[e] != INVALID) { time_us[e] = INVALID; ++counts[2]; } }
        }
    }
    if (mode == 2)
        for (int s = 0; s < NS; ++s) for (int k = 0; k < K; ++k) for (int p = 0; p < P; ++p)
            if (time_us[E(s, k, p)] != INVALID && int64_t(time_us[E(s, k, p)]) > threshold) { time_us[E(s, k, p)] = INVALID; ++counts[3]; }
    return 0;
}

}  // extern "C"
