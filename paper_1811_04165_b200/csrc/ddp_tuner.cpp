// The three tuners (host code): genetic algorithm over the joint chromosome of all pipeline kernels
// (settings BJ:cfg4), per-kernel exhaustive brute force and pure random search
// (P:221-223).  The fitness is either the CUDA-event harness of ddp_rt.cpp or a
// caller-supplied callback (tests, external drivers) -- the tuners never look inside it.
//
// Step-by-step specification: DESIGN.md "Tuners" (from SURVEY 8(c) GA/BF/random).  All randomness
// comes from one xoshiro256** stream per run, seeded from the run seed by splitmix64 and consumed in
// the order written here, so a run is a pure function of (seed, parameters, fitness values).
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstring>
#include <limits>

#include "ddp_internal.h"

namespace {
const double kInf = std::numeric_limits<double>::infinity();

struct Rng {
    uint64_t s[4];
    static uint64_t splitmix(uint64_t& x) {
        uint64_t z = (x += 0x9E3779B97F4A7C15ull);
        z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
        z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
        return z ^ (z >> 31);
    }
    explicit Rng(uint64_t seed) {
        uint64_t x = seed;
        for (int i = 0; i < 4; ++i) s[i] = splitmix(x);
    }
    static uint64_t rotl(uint64_t v, int k) { return (v << k) | (v >> (64 - k)); }
    uint64_t next() {
        const uint64_t r = rotl(s[1] * 5, 7) * 9, t = s[1] << 17;
        s[2] ^= s[0];
        s[3] ^= s[1];
        s[1] ^= s[2];
        s[0] ^= s[3];
        s[2] ^= t;
        s[3] = rotl(s[3], 45);
        return r;
    }
    int below(int n) { return (int)(((unsigned __int128)next() * (unsigned __int128)(uint64_t)n) >> 64); }  // [0, n)
    double unit() { return (double)(next() >> 11) * (1.0 / 9007199254740992.0); }                          // [0, 1)
};

struct Chrom {
    ddp_kcfg k[DDP_NSLOTS];
    double fit = kInf;
};
std::string chrom_key(const Chrom& c) { return std::string((const char*)c.k, sizeof c.k); }
bool chrom_equal(const Chrom& a, const Chrom& b) { return std::memcmp(a.k, b.k, sizeof a.k) == 0; }

double now_s() {
    return std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count();
}

// Shared bookkeeping of one tuning run: memoised fitness, evaluation counting, best-so-far history.
struct Run {
    ddp_plan* p;
    const ddp_tune_io* io;
    ddp_tune_result* res;
    bool hw;
    int64_t max_evals;
    std::unordered_map<std::string, double> memo;
    Chrom best;
    double best_per[DDP_NSLOTS] = {0, 0, 0, 0};
    int64_t compiles0;
    double t0;
    ddp_status err = DDP_OK;

    Run(ddp_plan* plan, const ddp_tune_io* tio, ddp_tune_result* r, int64_t cap)
        : p(plan), io(tio), res(r), hw(tio->fitness == nullptr), max_evals(cap) {
        compiles0 = ddp_rt_compile_count();
        t0 = now_s();
        res->n_fitness_calls = 0;
        res->n_kernel_timings = 0;
        res->n_compiles = 0;
        res->history_len = 0;
        res->best_ms = kInf;
        res->sum_isolated_min_ms = 0.0;
        for (int s = 0; s < DDP_NSLOTS; ++s) {
            res->kernel_ms[s] = 0.0;
            best.k[s] = canonical(s);
        }
    }
    // Value of an unused slot (direct plans have no sub2): the plan's default, never touched.
    ddp_kcfg canonical(int slot) const {
        const ddp_kernel k = ddp_slot_kernel(p, slot);
        return p->kcfg[k == DDP_K_COUNT ? DDP_K_SUB2 : k];
    }
    bool budget_left() const { return max_evals <= 0 || res->n_fitness_calls < max_evals; }

    // Raw fitness of a joint configuration; per[] = per-slot cost when the backend knows it.
    double raw(const ddp_kcfg cfg[DDP_NSLOTS], double per[DDP_NSLOTS], unsigned slot_mask, double best_so_far) {
        for (int s = 0; s < DDP_NSLOTS; ++s) per[s] = 0.0;
        if (!hw) return io->fitness(io->user, cfg);
        double ms = kInf;
        ddp_status st = ddp_rt_time_pipeline_mask(p, io, cfg, slot_mask, best_so_far, &ms, per, &res->n_kernel_timings);
        if (st != DDP_OK) err = st;
        return ms;
    }
    // Memoised evaluation; counts an evaluation only for a not-yet-seen chromosome.
    double eval(Chrom& c) {
        const std::string key = chrom_key(c);
        auto it = memo.find(key);
        if (it != memo.end()) return c.fit = it->second;
        double per[DDP_NSLOTS];
        const double f = raw(c.k, per, 0xFu, best.fit);
        record(c, f, per);
        memo[key] = f;
        return f;
    }
    void record(Chrom& c, double f, const double per[DDP_NSLOTS]) {
        c.fit = f;
        ++res->n_fitness_calls;
        if (f < best.fit) {
            best = c;
            for (int s = 0; s < DDP_NSLOTS; ++s) best_per[s] = per[s];
        }
        if (res->history && res->history_len < res->history_cap) res->history[res->history_len++] = best.fit;
    }
    // Compile every new code shape of the batch on all host cores before the (serial) timing.
    void precompile(const std::vector<Chrom>& batch) {
        if (!hw) return;
        std::vector<std::pair<ddp_kernel, ddp_kcfg>> list;
        for (const Chrom& c : batch) {
            if (memo.count(chrom_key(c))) continue;
            for (int s = 0; s < DDP_NSLOTS; ++s) {
                const ddp_kernel k = ddp_slot_kernel(p, s);
                if (k != DDP_K_COUNT) list.emplace_back(k, c.k[s]);
            }
        }
        ddp_rt_precompile(p, list);
    }
    // the configurations a run ends with (GA: last population, ranked; random: its last draws)
    void record_final(const std::vector<Chrom>& v) {
        res->final_len = 0;
        if (!res->final_pop || res->final_cap == 0) return;
        for (const Chrom& c : v) {
            if (res->final_len >= res->final_cap) break;
            for (int s = 0; s < DDP_NSLOTS; ++s) res->final_pop[res->final_len * DDP_NSLOTS + s] = c.k[s];
            if (res->final_fit) res->final_fit[res->final_len] = c.fit;
            ++res->final_len;
        }
    }
    ddp_status finish() {
        res->n_compiles = ddp_rt_compile_count() - compiles0;
        res->wall_seconds = now_s() - t0;
        if (err != DDP_OK) return err;
        if (res->n_fitness_calls == 0 || !(best.fit < kInf)) return ddp_fail(p, DDP_E_BUDGET, "no configuration evaluated successfully");
        res->best_ms = best.fit;
        for (int s = 0; s < DDP_NSLOTS; ++s) {
            res->best[s] = best.k[s];
            res->kernel_ms[s] = best_per[s];
            const ddp_kernel k = ddp_slot_kernel(p, s);
            if (k != DDP_K_COUNT) {
                ddp_status st = ddp_set_kcfg(p, k, &best.k[s]);
                if (st != DDP_OK) return st;
            }
        }
        return DDP_OK;
    }
};

// A3: every gene uniform over its candidate array, then repair (BJ:cfg4).
Chrom random_chrom(Run& R, Rng& rng) {
    Chrom c;
    const DdpGeneDomain* D = ddp_gene_domains();
    for (int s = 0; s < DDP_NSLOTS; ++s) {
        const ddp_kernel k = ddp_slot_kernel(R.p, s);
        if (k == DDP_K_COUNT) {
            c.k[s] = R.canonical(s);
            continue;
        }
        for (int g = 0; g < DDP_NGENES; ++g) *ddp_gene_ptr(&c.k[s], g) = D[g].v[rng.below(D[g].n)];
        ddp_repair_kcfg(R.p, k, &c.k[s]);
    }
    return c;
}

bool io_ok(const ddp_plan* p, const ddp_tune_io* io, const ddp_tune_result* res) {
    return p && io && res && (res->history == nullptr || res->history_cap > 0 || res->history_len == 0);
}
}  // namespace

// ------------------------------------------------------------------------------------ GA
extern "C" ddp_status ddp_tune_ga(ddp_plan* plan, const ddp_tune_io* io, const ddp_ga_params* gp, ddp_tune_result* res) {
    if (!io_ok(plan, io, res) || !gp) return DDP_E_ARG;
    if (plan->integ_mode != DDP_INTEG_DECIMATE) return ddp_fail(plan, DDP_E_CONFIG, "the tuners time the integrate and snr kernels: the plan must use DDP_INTEG_DECIMATE");
    const int N = gp->population, G = gp->generations, T = gp->tournament, E = gp->elitism;
    if (N < 2 || G < 0 || T < 1 || E < 0 || E >= N || !(gp->p_cross >= 0.0 && gp->p_cross <= 1.0) ||
        !(gp->p_mut >= 0.0 && gp->p_mut <= 1.0))
        return ddp_fail(plan, DDP_E_ARG, "GA parameters out of range");
    if (gp->max_evals < 0) return ddp_fail(plan, DDP_E_BUDGET, "negative evaluation budget");
    Run R(plan, io, res, gp->max_evals);
    Rng rng(gp->seed);
    const DdpGeneDomain* D = ddp_gene_domains();

    // A3: initial population
    std::vector<Chrom> pop(N);
    for (int i = 0; i < N; ++i) pop[i] = random_chrom(R, rng);
    R.precompile(pop);
    for (int i = 0; i < N && R.budget_left(); ++i) R.eval(pop[i]);

    auto rank = [](std::vector<Chrom>& v) {  // ascending fitness, ties keep index order
        std::stable_sort(v.begin(), v.end(), [](const Chrom& a, const Chrom& b) { return a.fit < b.fit; });
    };
    auto tournament = [&]() -> int {  // A5: best of T uniform draws with replacement, tie -> lower index
        int win = rng.below(N);
        for (int t = 1; t < T; ++t) {
            const int c = rng.below(N);
            if (pop[c].fit < pop[win].fit || (pop[c].fit == pop[win].fit && c < win)) win = c;
        }
        return win;
    };

    for (int gen = 0; gen < G && R.budget_left(); ++gen) {
        rank(pop);
        const int nchild = gp->replacement == 1 ? N : N - E;
        std::vector<Chrom> kids;
        kids.reserve(nchild + 1);
        while ((int)kids.size() < nchild) {
            const int ia = tournament();
            int ib = tournament();
            for (int tries = 0; tries < 8 && chrom_equal(pop[ia], pop[ib]); ++tries) ib = tournament();  // A6
            Chrom a = pop[ia], b = pop[ib];
            for (int s = 0; s < DDP_NSLOTS; ++s) {  // A7: per kernel with probability p_cross
                if (ddp_slot_kernel(plan, s) == DDP_K_COUNT) continue;
                if (!(rng.unit() < gp->p_cross)) continue;
                if (gp->crossover_kind == 1) {  // one-point (P:197a): genes after the cut are exchanged
                    const int cut = 1 + rng.below(DDP_NGENES - 1);
                    for (int g = cut; g < DDP_NGENES; ++g) std::swap(*ddp_gene_ptr(&a.k[s], g), *ddp_gene_ptr(&b.k[s], g));
                } else {  // coin toss (P:197b): exchange a gene when the random number exceeds 0.5
                    for (int g = 0; g < DDP_NGENES; ++g)
                        if (rng.unit() > 0.5) std::swap(*ddp_gene_ptr(&a.k[s], g), *ddp_gene_ptr(&b.k[s], g));
                }
            }
            Chrom* pair[2] = {&a, &b};
            for (Chrom* c : pair) {  // A8: new value differs from the old one
                for (int s = 0; s < DDP_NSLOTS; ++s) {
                    const ddp_kernel k = ddp_slot_kernel(plan, s);
                    if (k == DDP_K_COUNT) continue;
                    auto mutate_gene = [&](int g) {
                        if (D[g].n < 2) return;
                        const int old = ddp_gene_index(g, ddp_gene_get(c->k[s], g));
                        int nv = rng.below(D[g].n - 1);
                        if (nv >= old) ++nv;
                        *ddp_gene_ptr(&c->k[s], g) = D[g].v[nv];
                    };
                    if (gp->mutation_kind == 1) {  // paper: per kernel with probability p_mut, one gene
                        if (rng.unit() < gp->p_mut) mutate_gene(rng.below(DDP_NGENES));
                    } else {  // BJ:cfg4: per gene
                        for (int g = 0; g < DDP_NGENES; ++g)
                            if (rng.unit() < gp->p_mut) mutate_gene(g);
                    }
                    ddp_repair_kcfg(plan, k, &c->k[s]);  // A12 (BJ:cfg4)
                }
                c->fit = kInf;
            }
            kids.push_back(a);
            if ((int)kids.size() < nchild) kids.push_back(b);
        }
        R.precompile(kids);
        size_t evaluated = 0;
        for (; evaluated < kids.size(); ++evaluated) {
            if (!R.budget_left() && !R.memo.count(chrom_key(kids[evaluated]))) break;
            R.eval(kids[evaluated]);
        }
        kids.resize(evaluated);
        std::vector<Chrom> next;
        next.reserve(N);
        if (gp->replacement == 1) {  // best half of the parents and best half of the offspring
            rank(kids);
            const int keep_p = N - N / 2, keep_k = std::min<int>(N / 2, (int)kids.size());
            for (int i = 0; i < keep_p; ++i) next.push_back(pop[i]);
            for (int i = 0; i < keep_k; ++i) next.push_back(kids[i]);
        } else {  // BJ:cfg4: E elites unchanged (fitness reused) + offspring
            for (int i = 0; i < E; ++i) next.push_back(pop[i]);
            for (const Chrom& c : kids) next.push_back(c);
        }
        for (int i = 0; (int)next.size() < N; ++i) next.push_back(pop[i]);  // budget ran out mid-generation
        pop.swap(next);
    }
    rank(pop);
    R.record_final(pop);
    return R.finish();
}

// ------------------------------------------------------------------------------------ random search
extern "C" ddp_status ddp_tune_random(ddp_plan* plan, const ddp_tune_io* io, const ddp_rand_params* rp, ddp_tune_result* res) {
    if (!io_ok(plan, io, res) || !rp) return DDP_E_ARG;
    if (plan->integ_mode != DDP_INTEG_DECIMATE) return ddp_fail(plan, DDP_E_CONFIG, "the tuners time the integrate and snr kernels: the plan must use DDP_INTEG_DECIMATE");
    if (rp->max_evals <= 0) return ddp_fail(plan, DDP_E_BUDGET, "random search needs a positive evaluation budget");
    Run R(plan, io, res, rp->max_evals);
    Rng rng(rp->seed);
    int64_t stale = 0;  // consecutive draws that were already seen (tiny spaces)
    std::vector<Chrom> last;  // the newest evaluated draws, newest last
    while (R.budget_left() && stale < 100000) {
        const int64_t room = rp->max_evals - res->n_fitness_calls;
        std::vector<Chrom> batch((size_t)std::min<int64_t>(64, room));
        for (Chrom& c : batch) c = random_chrom(R, rng);
        R.precompile(batch);
        for (Chrom& c : batch) {
            if (!R.budget_left()) break;
            const int64_t before = res->n_fitness_calls;
            R.eval(c);
            stale = res->n_fitness_calls == before ? stale + 1 : 0;
            if (res->n_fitness_calls != before && res->final_pop && res->final_cap) {
                if (last.size() == res->final_cap) last.erase(last.begin());
                last.push_back(c);
            }
        }
    }
    R.record_final(last);
    return R.finish();
}

// ------------------------------------------------------------------------------------ brute force
// every kernel separately -- each valid configuration of kernel k is timed with the other
// kernels held at the plan's current (reference) configuration; the per-kernel winners are then timed
// together once, which is the figure comparable with the GA's joint fitness (GA.6).
extern "C" ddp_status ddp_tune_bruteforce(ddp_plan* plan, const ddp_tune_io* io, const ddp_bf_params* bp, ddp_tune_result* res) {
    if (!io_ok(plan, io, res) || !bp) return DDP_E_ARG;
    if (plan->integ_mode != DDP_INTEG_DECIMATE) return ddp_fail(plan, DDP_E_CONFIG, "the tuners time the integrate and snr kernels: the plan must use DDP_INTEG_DECIMATE");
    if (bp->max_evals_per_kernel < 0) return ddp_fail(plan, DDP_E_BUDGET, "negative evaluation budget");
    Run R(plan, io, res, 0);
    Chrom ref;
    for (int s = 0; s < DDP_NSLOTS; ++s) ref.k[s] = R.canonical(s);
    Chrom winners = ref;
    double per[DDP_NSLOTS];
    if (R.hw) R.raw(ref.k, per, 0xFu, kInf);  // one full pass so that every kernel's input buffer holds real data
    double sum_min = 0.0;
    for (int s = 0; s < DDP_NSLOTS; ++s) {
        const ddp_kernel k = ddp_slot_kernel(plan, s);
        if (k == DDP_K_COUNT) continue;
        if (bp->slots != 0 && !(bp->slots & (1u << s))) continue;
        const std::vector<ddp_kcfg>& V = ddp_valid_set(plan, k);
        size_t n = V.size(), stride = 1;
        if (bp->max_evals_per_kernel > 0 && (int64_t)n > bp->max_evals_per_kernel) {
            stride = (n + (size_t)bp->max_evals_per_kernel - 1) / (size_t)bp->max_evals_per_kernel;
        }
        double kbest = kInf, tbest = kInf;  // best kernel cost, and the total it was seen in (cut-off reference)
        for (size_t i0 = 0; i0 < n; i0 += 256 * stride) {  // batches: compile in parallel, then time
            std::vector<Chrom> batch;
            for (size_t i = i0; i < n && i < i0 + 256 * stride; i += stride) {
                Chrom c = ref;
                c.k[s] = V[i];
                batch.push_back(c);
            }
            R.precompile(batch);
            for (Chrom& c : batch) {
                const double total = R.raw(c.k, per, bp->isolated ? (1u << s) : 0xFu, tbest);
                const double cost = R.hw ? (std::isfinite(total) ? per[s] : kInf) : total;
                ++res->n_fitness_calls;
                if (cost < kbest) {
                    kbest = cost;
                    tbest = total;
                    winners.k[s] = c.k[s];
                }
                // history = the running sum of per-kernel minima found so far (kernels not yet searched
                // do not contribute), which is what "best so far" means for a per-kernel search
                if (res->history && res->history_len < res->history_cap)
                    res->history[res->history_len++] = sum_min + kbest;
            }
        }
        sum_min += kbest;
    }
    res->sum_isolated_min_ms = sum_min;
    // the four winners together (not counted as a search evaluation)
    const double joint = R.raw(winners.k, per, 0xFu, kInf);
    R.best = winners;
    R.best.fit = joint;
    for (int s = 0; s < DDP_NSLOTS; ++s) R.best_per[s] = per[s];
    return R.finish();
}

extern "C" ddp_status ddp_time_pipeline(ddp_plan* plan, const ddp_tune_io* io, const ddp_kcfg cfg[DDP_NSLOTS], double* ms,
                                        double kernel_ms[DDP_NSLOTS]) {
    if (!plan || !io || !cfg || !ms) return DDP_E_ARG;
    double per[DDP_NSLOTS] = {0, 0, 0, 0};
    ddp_status st = DDP_OK;
    if (io->fitness) {
        *ms = io->fitness(io->user, cfg);
    } else {
        int64_t nt = 0;
        st = ddp_rt_time_pipeline_mask(plan, io, cfg, 0xFu, kInf, ms, per, &nt);
    }
    if (kernel_ms)
        for (int s = 0; s < DDP_NSLOTS; ++s) kernel_ms[s] = per[s];
    return st;
}
