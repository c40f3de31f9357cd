// TEST INFRASTRUCTURE — NOT PART OF THE PRODUCT PATH.
//
// Plain, slow, obviously-correct CPU oracle for TANGRAM's pipeline-composition search
// (§5.2) as restated by BASELINE.json:north_star and SURVEY.md §8(c).
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
// call this.  It shares no code, header, table or constant generator with the CUDA library under
// paper_2606_16907_b200/csrc/ and neither includes the other.
//
// What is computed (SURVEY.md §8(c) "plain definition"):
//   plan  = stages (a_i,b_i,k_i), a_0=0, b_i=a_{i+1}, b_{n-1}=L, islands pairwise distinct,
//           c[a_i][b_i][k_i] finite                        (PAPER.md:51 cover; :260 subset of islands)
//   sum   = sum_i c[a_i][b_i][k_i] + sum_{i<n-1} x[k_i][k_{i+1}]     (PAPER.md:240 (1) activations cross)
//   T     = max_i c[a_i][b_i][k_i]                          (PAPER.md:250 (1) slowest stage = bottleneck)
//   iter  = sum + (m-1)*T                                   (north_star; 1F1B PAPER.md:248)
//   result= argmin of the key (iter, T, mask, k_0, b_0, k_1, b_1, ...)
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`):
//   orc_solve      : == orc_bruteforce (literal enumeration) on thousands of tiny instances, value and
//                    plan; closed forms K=1, m=1, identical islands; invariants; independent Python
//                    re-scorer; lane-less recurrence when all x are equal.
//   orc_reduce / x : hand-computed fixtures (tests/golden/) incl. A12's 64 MB @ 25/100/400 GB/s.
//   orc_prune      : brute-force O(P^2) dominance in Python, R1/R2 leave orc_solve unchanged, idempotent.
//   orc_bruteforce : is the definition itself; additionally pinned by hand-worked tiny cases.
// No function here is "parity unpinned".  (The paper prints no worked numeric example: Fig. 7 is
// missing from PAPER.md:242-244.)

#include <algorithm>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>

namespace {

constexpr int64_t INF = int64_t(1) << 30;       // saturating "no plan" (SURVEY.md §8 notation, A15)
constexpr int32_t INVALID = 0x7fffffff;         // "no such intra-slice plan" marker in time_us
constexpr int64_t TIME_MAX = int64_t(1) << 25;
constexpr int MAXK = 16;

struct Inst {
    int L, K, P, m;
    const int32_t* time_us;   // [NS][K][P]
    const int32_t* mem_mb;    // [NS][K][P]
    const int32_t* cap_mb;    // [K]
    const int32_t* bw_gbps;   // [K][K] sender-major
    int act_mb;
    int NS() const { return L * (L + 1) / 2; }
};

// slice index s(a,b), SURVEY.md §8 notation
inline int sidx(int L, int a, int b) { return a * (2 * L - a + 1) / 2 + (b - a - 1); }

struct Reduced {
    std::vector<int64_t> c;     // [NS][K], INF if no feasible plan
    std::vector<int32_t> argp;  // [NS][K], lowest p attaining c, -1 if none
    std::vector<int64_t> x;     // [K][K] sender j -> receiver k, 0 on the diagonal
};

// §8(a) step 1 (PAPER.md:240 "estimated execution times and memory requirements", :236 memory
// infeasibility) and step 2 (A12: x = ceil(act_mb*1000 / bw_gbps) microseconds).
Reduced reduce_tables(const Inst& I) {
    Reduced R;
    const int NS = I.NS(), K = I.K, P = I.P;
    R.c.assign(size_t(NS) * K, INF);
    R.argp.assign(size_t(NS) * K, -1);
    for (int s = 0; s < NS; ++s)
        for (int k = 0; k < K; ++k)
            for (int p = 0; p < P; ++p) {
                const size_t e = (size_t(s) * K + k) * P + p;
                if (I.time_us[e] == INVALID) continue;
                if (I.mem_mb[e] > I.cap_mb[k]) continue;
                if (int64_t(I.time_us[e]) < R.c[size_t(s) * K + k]) {   // strict: ties -> lowest p
                    R.c[size_t(s) * K + k] = I.time_us[e];
                    R.argp[size_t(s) * K + k] = p;
                }
            }
    R.x.assign(size_t(K) * K, 0);
    for (int j = 0; j < K; ++j)
        for (int k = 0; k < K; ++k) {
            if (j == k) continue;
            const int64_t num = int64_t(I.act_mb) * 1000, den = I.bw_gbps[j * K + k];
            int64_t v = (num + den - 1) / den;
            if (v > TIME_MAX) v = INF;                                  // edge unusable (§8(b) limits)
            R.x[size_t(j) * K + k] = v;
        }
    return R;
}

// §8(a) step 3 (PAPER.md:250 (1) "ranks the slowest stages"; A6): ascending distinct finite c.
std::vector<int64_t> candidates(const Reduced& R) {
    std::vector<int64_t> v;
    for (int64_t c : R.c) if (c < INF) v.push_back(c);
    std::sort(v.begin(), v.end());
    v.erase(std::unique(v.begin(), v.end()), v.end());
    return v;
}

inline int64_t sat(int64_t v) { return v >= INF ? INF : v; }

// One DP at threshold T (§8(c) algorithm step 3; PAPER.md:250 (2) front-first construction with
// memoisation; A1 laned state; A2 transfers do not count toward T).
//   g[a][S][k] = min cost of covering [a,L) with exactly the islands S, first stage on k, all stages <= T
//   h[b][R][k] = min_{j in R} x[k][j] + g[b][R][j]   (k not in R): transfer pre-minimum, §8(d)
struct DP {
    int L, K;
    std::vector<int32_t> g, h;
    std::vector<uint8_t> gb, hj;   // choices: next boundary b for g, next island j for h
    bool keep;
    size_t at(int a, uint32_t S, int k) const { return (size_t(S) * K + k) * (L + 1) + a; }
};

struct Top { int64_t best; uint32_t S; int k; };

Top run_dp(const Inst& I, const Reduced& R, int64_t T, DP& D, bool keep_choices) {
    const int L = I.L, K = I.K;
    const uint32_t NM = 1u << K;
    D.L = L; D.K = K; D.keep = keep_choices;
    D.g.assign(size_t(NM) * K * (L + 1), int32_t(INF));
    D.h.assign(size_t(NM) * K * (L + 1), int32_t(INF));
    if (keep_choices) { D.gb.assign(D.g.size(), 0); D.hj.assign(D.g.size(), 0); }
    for (int d = 1; d <= K; ++d) {
        // transfer pre-minimum for the wavefront below (masks Rm of size d-1)
        if (d >= 2)
            for (uint32_t Rm = 1; Rm < NM; ++Rm) {
                if (__builtin_popcount(Rm) != d - 1) continue;
                for (int k = 0; k < K; ++k) {
                    if (Rm >> k & 1) continue;
                    for (int b = 1; b < L; ++b) {
                        int64_t best = INF; int bj = 0;
                        for (int j = 0; j < K; ++j) {
                            if (!(Rm >> j & 1)) continue;
                            const int64_t v = sat(R.x[size_t(k) * K + j] + D.g[D.at(b, Rm, j)]);
                            if (v < best) { best = v; bj = j; }          // strict: ties -> lowest j
                        }
                        D.h[D.at(b, Rm, k)] = int32_t(best);
                        if (keep_choices) D.hj[D.at(b, Rm, k)] = uint8_t(bj);
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
                        const int64_t cv = R.c[size_t(sidx(L, a, b)) * K + k];
                        if (cv >= INF || cv > T) continue;               // infeasible or new bottleneck
                        int64_t cand;
                        if (b == L) cand = (Rm == 0) ? cv : INF;
                        else cand = (Rm == 0) ? INF : sat(cv + D.h[D.at(b, Rm, k)]);
                        if (cand < best) { best = cand; bb = b; }        // strict: ties -> lowest b
                    }
                    D.g[D.at(a, S, k)] = int32_t(best);
                    if (keep_choices) D.gb[D.at(a, S, k)] = uint8_t(bb);
                }
            }
        }
    }
    Top t{INF, 0, 0};
    for (uint32_t S = 1; S < NM; ++S)                                     // ties -> lowest S, lowest k
        for (int k = 0; k < K; ++k)
            if ((S >> k & 1) && D.g[D.at(0, S, k)] < t.best) t = Top{D.g[D.at(0, S, k)], S, k};
    return t;
}

}  // namespace

extern "C" {

struct orc_result {
    int64_t iter_time_us;     // INT64_MAX if infeasible
    int64_t sum_us;
    int64_t bottleneck_us;    // T*
    int32_t n_stages;
    uint32_t island_mask;
    int32_t n_dp_run;         // DPs executed (excluding the T=inf run and the final choice-keeping run)
    int32_t n_candidates;
    int32_t stage_begin[MAXK];
    int32_t stage_island[MAXK];
    int32_t stage_plan[MAXK];
};

static void set_infeasible(orc_result* o) {
    std::memset(o, 0, sizeof(*o));
    o->iter_time_us = INT64_MAX;
}

static void backtrack(const Inst& I, const Reduced& R, const DP& D, Top t, orc_result* o) {
    int a = 0, k = t.k; uint32_t S = t.S; int n = 0;
    while (true) {
        const int b = D.gb[D.at(a, S, k)];
        o->stage_begin[n] = a; o->stage_island[n] = k;
        o->stage_plan[n] = R.argp[size_t(sidx(I.L, a, b)) * I.K + k];
        ++n;
        if (b == I.L) break;
        const uint32_t Rm = S ^ (1u << k);
        const int j = D.hj[D.at(b, Rm, k)];
        a = b; S = Rm; k = j;
    }
    o->n_stages = n;
}

// DP at one threshold; T < 0 means T = infinity.  Writes f_T (INF=2^30 if infeasible), the argmin
// (S,k) and, if want_plan, the tie-broken plan at this T (iter/bottleneck fields: bottleneck = T given).
int orc_dp_at(int L, int K, int P, int m, const int32_t* time_us, const int32_t* mem_mb,
              const int32_t* cap_mb, const int32_t* bw_gbps, int act_mb, int64_t T, int want_plan,
              orc_result* out) {
    Inst I{L, K, P, m, time_us, mem_mb, cap_mb, bw_gbps, act_mb};
    Reduced R = reduce_tables(I);
    DP D;
    const int64_t Teff = T < 0 ? INF : T;
    Top t = run_dp(I, R, Teff, D, want_plan != 0);
    set_infeasible(out);
    if (t.best >= INF) return 0;
    out->sum_us = t.best; out->island_mask = t.S; out->bottleneck_us = Teff;
    out->iter_time_us = t.best + int64_t(m - 1) * Teff;
    out->stage_island[0] = t.k;
    if (want_plan) backtrack(I, R, D, t, out);
    return 0;
}

// Full solve (§8(c) steps 1-5).  full_sweep != 0: run every candidate (no bisection, no stop rule A7).
// n_threads > 1: candidates are evaluated in blocks of n_threads independent DP(T) calls and folded in
// ascending order with the same rules, so the result is identical to the sequential sweep.
int orc_solve(int L, int K, int P, int m, const int32_t* time_us, const int32_t* mem_mb,
              const int32_t* cap_mb, const int32_t* bw_gbps, int act_mb, int full_sweep, int n_threads,
              orc_result* out) {
    Inst I{L, K, P, m, time_us, mem_mb, cap_mb, bw_gbps, act_mb};
    Reduced R = reduce_tables(I);
    std::vector<int64_t> cand = candidates(R);
    set_infeasible(out);
    out->n_candidates = int(cand.size());
    DP D0;
    const Top tinf = run_dp(I, R, INF, D0, false);                       // step 4: f_inf
    if (tinf.best >= INF) return 0;
    const int64_t f_inf = tinf.best;
    const int n = int(cand.size());
    if (n_threads < 1) n_threads = 1;

    auto eval_block = [&](int i0, int cnt, std::vector<Top>& res) {
        res.assign(cnt, Top{INF, 0, 0});
        std::vector<std::thread> th;
        for (int t = 0; t < cnt; ++t)
            th.emplace_back([&, t] { DP D; res[t] = run_dp(I, R, cand[i0 + t], D, false); });
        for (auto& x : th) x.join();
    };

    int lo = 0;
    int n_dp = 0;
    if (!full_sweep) {
        // feasibility is monotone in T (a plan admissible at T stays admissible at T' > T):
        // bisection for the lowest feasible candidate; cand[n-1] is feasible because f_inf is finite.
        int l = 0, r = n - 1;
        while (l < r) {
            const int mid = (l + r) / 2;
            DP D; ++n_dp;
            if (run_dp(I, R, cand[mid], D, false).best < INF) r = mid; else l = mid + 1;
        }
        lo = l;
    }
    bool have = false; int64_t best_iter = 0, best_T = 0;
    std::vector<Top> res;
    for (int i0 = lo; i0 < n; i0 += n_threads) {
        const int cnt = std::min(n_threads, n - i0);
        bool stop = false;
        if (!full_sweep && have && f_inf + int64_t(m - 1) * cand[i0] >= best_iter) break;   // A7
        eval_block(i0, cnt, res);
        for (int t = 0; t < cnt; ++t) {
            const int64_t T = cand[i0 + t];
            if (!full_sweep && have && f_inf + int64_t(m - 1) * T >= best_iter) { stop = true; break; }
            ++n_dp;
            if (res[t].best >= INF) continue;
            const int64_t it = res[t].best + int64_t(m - 1) * T;
            if (!have || it < best_iter) { have = true; best_iter = it; best_T = T; }   // ties keep lower T
        }
        if (stop) break;
    }
    // step 5: re-run at T* keeping choices, back-track
    DP D;
    const Top t = run_dp(I, R, best_T, D, true);
    out->iter_time_us = best_iter; out->sum_us = t.best; out->bottleneck_us = best_T;
    out->island_mask = t.S; out->n_dp_run = n_dp;
    backtrack(I, R, D, t, out);
    return 0;
}

// §8(c) step 6: literal enumeration of the plain definition.
namespace {
struct BF {
    const Inst* I; const Reduced* R;
    std::vector<int64_t> bestkey; bool have = false;
    std::vector<int> seq;  // k_0,b_0,k_1,b_1,...
    int64_t n_plans = 0;
    void rec(int a, uint32_t used, int prev, int64_t sum, int64_t T) {
        const int L = I->L, K = I->K;
        if (a == L) {
            ++n_plans;
            std::vector<int64_t> key{sum + int64_t(I->m - 1) * T, T, int64_t(used)};
            for (int v : seq) key.push_back(v);
            if (!have || key < bestkey) { have = true; bestkey = key; }
            return;
        }
        for (int k = 0; k < K; ++k) {
            if (used >> k & 1) continue;
            for (int b = a + 1; b <= L; ++b) {
                const int64_t cv = R->c[size_t(sidx(L, a, b)) * K + k];
                if (cv >= INF) continue;
                int64_t xs = 0;
                if (prev >= 0) { xs = R->x[size_t(prev) * K + k]; if (xs >= INF) continue; }
                seq.push_back(k); seq.push_back(b);
                rec(b, used | (1u << k), k, sum + cv + xs, std::max(T, cv));
                seq.pop_back(); seq.pop_back();
            }
        }
    }
};
}  // namespace

int orc_bruteforce(int L, int K, int P, int m, const int32_t* time_us, const int32_t* mem_mb,
                   const int32_t* cap_mb, const int32_t* bw_gbps, int act_mb, orc_result* out,
                   int64_t* n_plans_out) {
    Inst I{L, K, P, m, time_us, mem_mb, cap_mb, bw_gbps, act_mb};
    Reduced R = reduce_tables(I);
    BF bf; bf.I = &I; bf.R = &R;
    bf.rec(0, 0, -1, 0, 0);
    set_infeasible(out);
    if (n_plans_out) *n_plans_out = bf.n_plans;
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
        out->stage_plan[i] = R.argp[size_t(sidx(L, a, b)) * K + k];
        a = b;
    }
    return 0;
}

// Second, independent recurrence (SURVEY.md §8(c) pins): when every off-diagonal x equals one value
// xc, the boundary-island lane is redundant and a lane-less (a,S) DP gives the optimum iteration
// time.  Returns min over T of f_T + (m-1)T via full sweep, or INT64_MAX.  xc is passed by the test.
int64_t orc_laneless_iter(int L, int K, int P, int m, const int32_t* time_us, const int32_t* mem_mb,
                          const int32_t* cap_mb, int64_t xc) {
    Inst I{L, K, P, m, time_us, mem_mb, cap_mb, nullptr, 0};
    const int NS = I.NS();
    std::vector<int64_t> c(size_t(NS) * K, INF);
    for (int s = 0; s < NS; ++s) for (int k = 0; k < K; ++k) for (int p = 0; p < P; ++p) {
        const size_t e = (size_t(s) * K + k) * P + p;
        if (time_us[e] != INVALID && mem_mb[e] <= cap_mb[k]) c[size_t(s) * K + k] = std::min<int64_t>(c[size_t(s) * K + k], time_us[e]);
    }
    std::vector<int64_t> cand;
    for (int64_t v : c) if (v < INF) cand.push_back(v);
    std::sort(cand.begin(), cand.end());
    int64_t best = INT64_MAX;
    const uint32_t NM = 1u << K;
    for (int64_t T : cand) {
        // w[a][S]: min cost to cover [a,L) using exactly S (any order); w[L][0] = -xc so that the
        // last stage pays no transfer
        std::vector<int64_t> w(size_t(L + 1) * NM, INF * 64);
        w[size_t(L) * NM + 0] = -xc;
        for (int a = L - 1; a >= 0; --a)
            for (uint32_t S = 1; S < NM; ++S)
                for (int k = 0; k < K; ++k) {
                    if (!(S >> k & 1)) continue;
                    for (int b = a + 1; b <= L; ++b) {
                        const int64_t cv = c[size_t(sidx(L, a, b)) * K + k];
                        if (cv >= INF || cv > T) continue;
                        const int64_t r = w[size_t(b) * NM + (S ^ (1u << k))];
                        if (r >= INF * 32) continue;
                        w[size_t(a) * NM + S] = std::min(w[size_t(a) * NM + S], cv + xc + r);
                    }
                }
        for (uint32_t S = 1; S < NM; ++S)
            if (w[S] < INF * 32) best = std::min(best, w[S] + int64_t(m - 1) * T);
    }
    return best;
}

// Reduced tables, for direct pinning of steps 1-3.  c_out [NS][K] int64 (2^30 = none), argp_out [NS][K]
// (-1 = none), x_out [K][K] int64; cand_out capacity NS*K, returns the candidate count.
int orc_reduce(int L, int K, int P, const int32_t* time_us, const int32_t* mem_mb, const int32_t* cap_mb,
               const int32_t* bw_gbps, int act_mb, int64_t* c_out, int32_t* argp_out, int64_t* x_out,
               int64_t* cand_out) {
    Inst I{L, K, P, 1, time_us, mem_mb, cap_mb, bw_gbps, act_mb};
    Reduced R = reduce_tables(I);
    std::copy(R.c.begin(), R.c.end(), c_out);
    std::copy(R.argp.begin(), R.argp.end(), argp_out);
    std::copy(R.x.begin(), R.x.end(), x_out);
    std::vector<int64_t> cd = candidates(R);
    std::copy(cd.begin(), cd.end(), cand_out);
    return int(cd.size());
}

// tg_prune oracle (§8(c) rules R1-R4; PAPER.md:234-236 policies, :43/:360 incompatible plans).
// mode 0: R1+R2; 1: +R3 (threshold = theta per mille, 1000..16384); 2: +R4 (threshold = cap in us).
// time_us is modified in place (dead := INVALID); counts[4] = entries newly killed by R1..R4.
int orc_prune(int L, int K, int P, int32_t* time_us, const int32_t* mem_mb, const int32_t* cap_mb,
              int mode, int64_t threshold, int64_t* counts) {
    const int NS = L * (L + 1) / 2;
    counts[0] = counts[1] = counts[2] = counts[3] = 0;
    auto E = [&](int s, int k, int p) { return (size_t(s) * K + k) * P + p; };
    // R1 infeasible
    for (int s = 0; s < NS; ++s) for (int k = 0; k < K; ++k) for (int p = 0; p < P; ++p)
        if (time_us[E(s, k, p)] != INVALID && mem_mb[E(s, k, p)] > cap_mb[k]) { time_us[E(s, k, p)] = INVALID; ++counts[0]; }
    // R2 dominated inside one (slice, island) cell on (time, memory).  Decided on
    // the cell as it stood before R2 (dominance is transitive, so this equals sequential removal).
    for (int s = 0; s < NS; ++s) for (int k = 0; k < K; ++k) {
        std::vector<char> dead(P, 0);
        for (int p = 0; p < P; ++p) {
            if (time_us[E(s, k, p)] == INVALID) continue;
            const int64_t tp = time_us[E(s, k, p)], mp = mem_mb[E(s, k, p)];
            for (int q = 0; q < P; ++q) {
                if (q == p || time_us[E(s, k, q)] == INVALID) continue;
                const int64_t tq = time_us[E(s, k, q)], mq = mem_mb[E(s, k, q)];
                if ((tq < tp && mq <= mp) || (tq <= tp && mq < mp) || (tq == tp && mq == mp && q < p)) dead[p] = 1;
            }
        }
        for (int p = 0; p < P; ++p) if (dead[p]) { time_us[E(s, k, p)] = INVALID; ++counts[1]; }
    }
    if (mode == 1) {
        // R3 imbalance: capacity from profiled atom throughput, demand = number of atoms
        std::vector<int64_t> C(K, 0); int64_t Ct = 0;
        for (int k = 0; k < K; ++k) {
            int64_t tau = 0; bool ok = true;
            for (int l = 0; l < L; ++l) {
                int64_t best = INF;
                for (int p = 0; p < P; ++p) { const int32_t t = time_us[E(sidx(L, l, l + 1), k, p)]; if (t != INVALID) best = std::min<int64_t>(best, t); }
                if (best >= INF) { ok = false; break; }
                tau += best;
            }
            if (ok) { if (tau < 1) tau = 1; C[k] = (int64_t(1) << 32) / tau; Ct += C[k]; }
        }
        for (int a = 0; a < L; ++a) for (int b = a + 1; b <= L; ++b) for (int k = 0; k < K; ++k) {
            if (C[k] == 0) continue;                                       // exempt
            const int64_t len = b - a;
            const bool over = len * Ct * 1000 > threshold * C[k] * L;
            const bool under = len * Ct * threshold < int64_t(1000) * C[k] * L;
            if (!(over || under)) continue;
            for (int p = 0; p < P; ++p) { const size_t e = E(sidx(L, a, b), k, p); if (time_us[e] != INVALID) { time_us[e] = INVALID; ++counts[2]; } }
        }
    }
    if (mode == 2) {
        for (int s = 0; s < NS; ++s) for (int k = 0; k < K; ++k) for (int p = 0; p < P; ++p)
            if (time_us[E(s, k, p)] != INVALID && int64_t(time_us[E(s, k, p)]) > threshold) { time_us[E(s, k, p)] = INVALID; ++counts[3]; }
    }
    return 0;
}

int orc_hw_threads() { return int(std::thread::hardware_concurrency()); }

}  // extern "C"
