// TEST INFRASTRUCTURE — NOT PART OF THE PRODUCT PATH.
//
// CPU oracle for SURVEY.md §8(f) NEXT-2: multi-stage partial plans.  PAPER.md:163 "a model-slice/island plan can
// include multiple pipeline stages"; :248 "model-slice/island plans themselves can contain several pipeline stages
// depending on the output of the LLM parallelizer"; :250 (1) "it ranks the slowest stages in all model-slice/island
// plans" -- the bottleneck of a partial plan is its SLOWEST INTERNAL STAGE, not its whole execution time.
// Separate translation unit: the core oracle and the depth / transfer-bound unit stay untouched.  Shares no code with
// the CUDA library.
//
// Model (reading N2).  Every table entry e = (slice, island k, intra-slice plan p) carries
//     time_us[e]   execution time of the whole partial plan for one microbatch = the sum over its internal stages
//                  (what the core path calls the stage time),
//     slow_us[e]   its slowest internal stage, 0 <= slow_us <= time_us,
//     q[e]         its number of internal pipeline stages, >= 1 (reported; does not enter the optimum),
//     mem_mb[e]    static memory, feasible iff mem_mb <= cap_mb[k] (the core rule).
// A plan is a sequence of partial plans (a_i, b_i, k_i, p_i) tiling [0, L) on pairwise distinct islands, every entry
// valid and feasible.  With x the transfer times of the core path,
//     sum  = sum_i time[e_i] + sum_i x[k_i][k_{i+1}]
//     T    = max_i slow[e_i]                  (the pipeline's slowest stage, PAPER.md:250 (1))
//     iter = sum + (m - 1) * T                (1F1B: one pass through every stage, then m - 1 beats of the slowest)
// and the result is the plan minimising the key (iter, T, mask, k_0, b_0, ..., k_{n-1}, b_{n-1}, p_0, ..., p_{n-1}).
// Equivalent threshold form (what the DP computes): at threshold T an entry is admissible iff slow <= T, the cost of a
// (slice, island) cell is c_T = min time over its admissible feasible entries (ties -> lowest p) -- a step function of T
// per cell --, f_T = the core recurrence on c_T, iter = min over candidate T of f_T + (m-1) T, candidates = the distinct
// slow values of the valid feasible entries.  At the optimum T* = max_i slow[e_i] (a plan admissible at T* whose slowest
// stage were lower would win at that lower candidate), and p_i = lowest p attaining c_{T*} of its cell.
// With slow == time everywhere this is the core definition bit for bit.
//
// Pins (tests/test_oracle_stages.py, all -m "not gpu"): orc_stages_solve == orc_stages_bruteforce (literal enumeration
// over cut sets, ordered island subsets AND plan choices) on thousands of tiny instances; slow == time reproduces the
// core oracle (value and plan); a hand-worked two-plan case where the lower-sum plan has the slower internal stage;
// lowering slow values never worsens the optimum; the reported T* is the largest slow of the returned plan; an
// independent re-scorer from the raw tables.

#include <algorithm>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

constexpr int64_t INF = int64_t(1) << 30;
constexpr int32_t INVALID = 0x7fffffff;
constexpr int64_t TIME_MAX = int64_t(1) << 25;
constexpr int MAXK = 16;

struct Inst {
    int L, K, P, m;
    const int32_t *time_us, *mem_mb, *slow_us, *q_stages, *cap_mb, *bw_gbps;   // q_stages may be null (= ones)
    int act_mb;
    int NS() const { return L * (L + 1) / 2; }
};

inline int sidx(int L, int a, int b) { return a * (2 * L - a + 1) / 2 + (b - a - 1); }
inline int64_t sat(int64_t v) { return v >= INF ? INF : v; }

// cost of cell (s, k) at threshold T: min time over valid feasible entries with slow <= T, ties -> lowest p
inline int64_t cost_at(const Inst& I, int s, int k, int64_t T, int* p_out) {
    int64_t best = INF; int bp = -1;
    for (int p = 0; p < I.P; ++p) {
        const size_t e = (size_t(s) * I.K + k) * I.P + p;
        if (I.time_us[e] == INVALID) continue;
        if (I.mem_mb[e] > I.cap_mb[k]) continue;
        if (int64_t(I.slow_us[e]) > T) continue;
        if (int64_t(I.time_us[e]) < best) { best = I.time_us[e]; bp = p; }   // strict: lowest p
    }
    if (p_out) *p_out = bp;
    return best;
}

std::vector<int64_t> transfers(const Inst& I) {
    std::vector<int64_t> x(size_t(I.K) * I.K, 0);
    for (int j = 0; j < I.K; ++j)
        for (int k = 0; k < I.K; ++k) {
            if (j == k) continue;
            const int64_t num = int64_t(I.act_mb) * 1000, den = I.bw_gbps[j * I.K + k];
            int64_t v = (num + den - 1) / den;
            if (v > TIME_MAX) v = INF;
            x[size_t(j) * I.K + k] = v;
        }
    return x;
}

std::vector<int64_t> candidates(const Inst& I) {
    std::vector<int64_t> v;
    const int NS = I.NS();
    for (int s = 0; s < NS; ++s)
        for (int k = 0; k < I.K; ++k)
            for (int p = 0; p < I.P; ++p) {
                const size_t e = (size_t(s) * I.K + k) * I.P + p;
                if (I.time_us[e] != INVALID && I.mem_mb[e] <= I.cap_mb[k]) v.push_back(I.slow_us[e]);
            }
    std::sort(v.begin(), v.end());
    v.erase(std::unique(v.begin(), v.end()), v.end());
    return v;
}

struct DP {
    int L, K;
    std::vector<int32_t> g, h;
    std::vector<uint8_t> gb, hj;
    size_t at(int a, uint32_t S, int k) const { return (size_t(S) * K + k) * (L + 1) + a; }
};
struct Top { int64_t best; uint32_t S; int k; };

// The core recurrence (front-first, laned state) on the costs c_T of this threshold.
Top run_dp(const Inst& I, const std::vector<int64_t>& x, int64_t T, DP& D, bool keep) {
    const int L = I.L, K = I.K, NS = I.NS();
    const uint32_t NM = 1u << K;
    std::vector<int64_t> c(size_t(NS) * K);
    for (int s = 0; s < NS; ++s) for (int k = 0; k < K; ++k) c[size_t(s) * K + k] = cost_at(I, s, k, T, nullptr);
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
                            const int64_t v = sat(x[size_t(k) * K + j] + D.g[D.at(b, Rm, j)]);
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
                        const int64_t cv = c[size_t(sidx(L, a, b)) * K + k];
                        if (cv >= INF) continue;                          // no admissible entry at this threshold
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

// Ascending sweep over the candidate thresholds with the exact stop rule f_inf + (m-1) T >= incumbent, then a
// choice-keeping run at T* and the back-track.  *pipeline_stages_out (may be null) = total number of pipeline stages of
// the returned plan, the sum of q over its partial plans.
int orc_stages_solve(int L, int K, int P, int m, const int32_t* time_us, const int32_t* mem_mb, const int32_t* slow_us,
                     const int32_t* q_stages, const int32_t* cap_mb, const int32_t* bw_gbps, int act_mb, orc_result* out,
                     int32_t* pipeline_stages_out) {
    Inst I{L, K, P, m, time_us, mem_mb, slow_us, q_stages, cap_mb, bw_gbps, act_mb};
    const std::vector<int64_t> x = transfers(I);
    const std::vector<int64_t> cand = candidates(I);
    set_infeasible(out);
    if (pipeline_stages_out) *pipeline_stages_out = 0;
    out->n_candidates = int(cand.size());
    DP D0;
    const Top tinf = run_dp(I, x, INF, D0, false);
    if (tinf.best >= INF) return 0;
    bool have = false; int64_t best_iter = 0, best_T = 0; int n_dp = 0;
    for (int64_t T : cand) {
        if (have && tinf.best + int64_t(m - 1) * T >= best_iter) break;
        DP D; ++n_dp;
        const Top t = run_dp(I, x, T, D, false);
        if (t.best >= INF) continue;
        const int64_t it = t.best + int64_t(m - 1) * T;
        if (!have || it < best_iter) { have = true; best_iter = it; best_T = T; }    // ties keep the lower T
    }
    DP D;
    const Top t = run_dp(I, x, best_T, D, true);
    out->iter_time_us = best_iter; out->sum_us = t.best; out->bottleneck_us = best_T;
    out->island_mask = t.S; out->n_dp_run = n_dp;
    int a = 0, k = t.k, n = 0, total_q = 0; uint32_t S = t.S;
    while (true) {
        const int b = D.gb[D.at(a, S, k)];
        int p = -1;
        cost_at(I, sidx(L, a, b), k, best_T, &p);
        out->stage_begin[n] = a; out->stage_island[n] = k; out->stage_plan[n] = p;
        total_q += q_stages ? q_stages[(size_t(sidx(L, a, b)) * K + k) * P + p] : 1;
        ++n;
        if (b == L) break;
        const uint32_t Rm = S ^ (1u << k);
        const int j = D.hj[D.at(b, Rm, k)];
        a = b; S = Rm; k = j;
    }
    out->n_stages = n;
    if (pipeline_stages_out) *pipeline_stages_out = total_q;
    return 0;
}

// Literal enumeration of the definition: every cut set, every ordered choice of distinct islands, every choice of plans.
namespace {
struct BF {
    const Inst* I; const std::vector<int64_t>* x;
    std::vector<int64_t> bestkey; bool have = false;
    std::vector<int> ks, bs, ps;
    int64_t n_plans = 0;
    void rec(int a, uint32_t used, int prev, int64_t sum, int64_t T) {
        const int L = I->L, K = I->K, P = I->P;
        if (a == L) {
            ++n_plans;
            std::vector<int64_t> key{sum + int64_t(I->m - 1) * T, T, int64_t(used)};
            for (size_t i = 0; i < ks.size(); ++i) { key.push_back(ks[i]); key.push_back(bs[i]); }
            for (int p : ps) key.push_back(p);
            if (!have || key < bestkey) { have = true; bestkey = key; }
            return;
        }
        for (int k = 0; k < K; ++k) {
            if (used >> k & 1) continue;
            int64_t xs = 0;
            if (prev >= 0) { xs = (*x)[size_t(prev) * K + k]; if (xs >= INF) continue; }
            for (int b = a + 1; b <= L; ++b)
                for (int p = 0; p < P; ++p) {
                    const size_t e = (size_t(sidx(L, a, b)) * K + k) * P + p;
                    if (I->time_us[e] == INVALID || I->mem_mb[e] > I->cap_mb[k]) continue;
                    ks.push_back(k); bs.push_back(b); ps.push_back(p);
                    rec(b, used | (1u << k), k, sum + I->time_us[e] + xs, std::max<int64_t>(T, I->slow_us[e]));
                    ks.pop_back(); bs.pop_back(); ps.pop_back();
                }
        }
    }
};
}  // namespace

int orc_stages_bruteforce(int L, int K, int P, int m, const int32_t* time_us, const int32_t* mem_mb, const int32_t* slow_us,
                          const int32_t* q_stages, const int32_t* cap_mb, const int32_t* bw_gbps, int act_mb, orc_result* out,
                          int32_t* pipeline_stages_out, int64_t* n_plans_out) {
    Inst I{L, K, P, m, time_us, mem_mb, slow_us, q_stages, cap_mb, bw_gbps, act_mb};
    const std::vector<int64_t> x = transfers(I);
    BF bf; bf.I = &I; bf.x = &x;
    bf.rec(0, 0, -1, 0, 0);
    set_infeasible(out);
    if (pipeline_stages_out) *pipeline_stages_out = 0;
    if (n_plans_out) *n_plans_out = bf.n_plans;
    if (!bf.have) return 0;
    out->iter_time_us = bf.bestkey[0]; out->bottleneck_us = bf.bestkey[1];
    out->island_mask = uint32_t(bf.bestkey[2]);
    out->sum_us = bf.bestkey[0] - int64_t(m - 1) * bf.bestkey[1];
    const int n = int(bf.bestkey.size() - 3) / 3;
    out->n_stages = n;
    int a = 0, total_q = 0;
    for (int i = 0; i < n; ++i) {
        const int k = int(bf.bestkey[3 + 2 * i]), b = int(bf.bestkey[4 + 2 * i]), p = int(bf.bestkey[3 + 2 * n + i]);
        out->stage_begin[i] = a; out->stage_island[i] = k; out->stage_plan[i] = p;
        total_q += q_stages ? q_stages[(size_t(sidx(L, a, b)) * K + k) * P + p] : 1;
        a = b;
    }
    if (pipeline_stages_out) *pipeline_stages_out = total_q;
    return 0;
}

}  // extern "C"
