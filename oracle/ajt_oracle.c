/*
 * ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU statement of what the hot path computes, written from
 * /root/reference/PAPER.md (cited as PAPER.md:N) and the readings listed in DESIGN.md ("Readings").
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * load this file.  It shares no code, header, table or helper with paper_2606_04484_b200/csrc/.
 *
 *   - merge        : the DEFINITION, by brute-force pairwise prefix comparison (no hashing, no sorting).
 *   - block merge  : Algorithm 1 line by line on timelines of message blocks (Match = text | token).
 *   - loss         : fp64 throughout, from the exact stored input values (steps 1-7; steps 8-9 in the extended entry).
 * (oracle/__init__.py adds, in plain numpy: pack_loss_inputs, the next-token alignment sequence by sequence, and
 *  lm_head_logp, log-probs / entropy from hidden states with an fp64 matmul as a library step.)
 *
 * Parity status: every function here and in oracle/__init__.py is pinned by tests/test_oracle_*.py (hand traces of
 * Algorithm 1 on tokens and on blocks, second independent formulations, invariants, closed forms, finite differences,
 * torch fp64 autograd, library routines).  Nothing is "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o oracle/libajt_oracle.so oracle/ajt_oracle.c -lm
 * OpenMP only parallelises independent outer loops (timelines j, rows t); no blocking, fusion or
 * reordering of the arithmetic inside one timeline pair or one row.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OWNER_LONGEST 0
#define ORACLE_OWNER_PAPER 1

/* i extends j  <=>  same group, i > j, L_i >= L_j, x_i[p] == x_j[p] for all p < L_j.
 * PAPER.md:182 ("mergeable when |S| >= |T| and Match(S[k],T[k]) for all k in [1,|T|]"),
 * PAPER.md:197-204 (Alg. 1 inner loop: j runs over earlier indices only),
 * PAPER.md:233 (token strategy: exact token-id match at every aligned position). */
static int extends(const int32_t* tokens, const int64_t* offsets, const int32_t* traj_ids, int64_t i, int64_t j) {
    if (!(i > j)) return 0;
    if (traj_ids[i] != traj_ids[j]) return 0;
    int64_t Li = offsets[i + 1] - offsets[i], Lj = offsets[j + 1] - offsets[j];
    if (Li < Lj) return 0;
    const int32_t* xi = tokens + offsets[i];
    const int32_t* xj = tokens + offsets[j];
    for (int64_t p = 0; p < Lj; ++p)
        if (xi[p] != xj[p]) return 0;
    return 1;
}

static int mask_at(const int32_t* resp_start, const uint8_t* mask_in, const int64_t* offsets, int64_t j, int64_t p) {
    if (mask_in) return mask_in[offsets[j] + p] != 0;
    return p >= (int64_t)resp_start[j];
}

/*
 * Merge oracle.  Returns 0, or -1 on invalid input (n < 0, zero-length timeline,
 * non-monotone offsets, unknown owner rule).
 *
 * Outputs (caller-allocated, worst-case capacity N_in tokens / n sequences):
 *   merged_tokens[N_out], merged_mask[N_out], merged_src[N_out], merged_old_logp[N_out] (may be NULL),
 *   merged_offsets[M+1], merged_origin[M], merged_traj[M], owner[n], counts[2] = {M, N_out}.
 */
int ajt_oracle_merge(const int32_t* tokens, const int64_t* offsets, const int32_t* traj_ids,
                     const int32_t* resp_start, const uint8_t* mask_in, const float* old_logp_in,
                     int32_t n, int32_t owner_rule,
                     int32_t* merged_tokens, uint8_t* merged_mask, int32_t* merged_src, float* merged_old_logp,
                     int64_t* merged_offsets, int32_t* merged_origin, int32_t* merged_traj,
                     int32_t* owner, int64_t* counts) {
    if (n < 0) return -1;
    if (owner_rule != ORACLE_OWNER_LONGEST && owner_rule != ORACLE_OWNER_PAPER) return -1;
    if (!resp_start && !mask_in) return -1;
    if (offsets[0] != 0) return -1;
    for (int64_t j = 0; j < n; ++j)
        if (offsets[j + 1] - offsets[j] < 1) return -1; /* L_j >= 1 (a message has BoS..EoS) */

    uint8_t* survives = (uint8_t*)malloc((size_t)n + 1);
    int64_t* last_ext = (int64_t*)malloc(sizeof(int64_t) * ((size_t)n + 1));
    int64_t* owner_tl = (int64_t*)malloc(sizeof(int64_t) * ((size_t)n + 1));
    int64_t* midx = (int64_t*)malloc(sizeof(int64_t) * ((size_t)n + 1));

    /* Step 2. Survivors: j survives <=> no i extends j.  (Alg. 1 removes every absorbed j,
     * PAPER.md:221-228.)  last_ext[j] = max{i : i extends j}. */
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t j = 0; j < n; ++j) {
        int64_t le = -1;
        for (int64_t i = j + 1; i < n; ++i)
            if (extends(tokens, offsets, traj_ids, i, j)) le = i;
        last_ext[j] = le;
        survives[j] = (le < 0);
    }

    /* Step 3. Owner. */
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t j = 0; j < n; ++j) {
        if (survives[j]) { owner_tl[j] = j; continue; }
        if (owner_rule == ORACLE_OWNER_PAPER) {
            /* Algorithm 1 taken literally: reverse order => the latest extender absorbs
             * (PAPER.md:178, 189-227). */
            owner_tl[j] = last_ext[j];
        } else {
            /* BASELINE.json north_star: "the longest extender wins, then the lowest index";
             * candidates restricted to survivors (reading M-3). */
            int64_t best = -1, bestL = -1;
            for (int64_t i = j + 1; i < n; ++i) {
                if (!survives[i]) continue;
                if (!extends(tokens, offsets, traj_ids, i, j)) continue;
                int64_t Li = offsets[i + 1] - offsets[i];
                if (Li > bestL) { bestL = Li; best = i; } /* ascending i: first of equal length is lowest */
            }
            owner_tl[j] = best; /* never -1: last_ext[j] survives (lemma, tested) */
        }
    }

    /* Survivors numbered in ascending original index ("in original order"). */
    int64_t M = 0, Nout = 0;
    for (int64_t j = 0; j < n; ++j) {
        if (survives[j]) {
            midx[j] = M;
            merged_origin[M] = (int32_t)j;
            merged_traj[M] = traj_ids[j];
            merged_offsets[M] = Nout;
            Nout += offsets[j + 1] - offsets[j];
            ++M;
        } else {
            midx[j] = -1;
        }
    }
    merged_offsets[M] = Nout;
    counts[0] = M;
    counts[1] = Nout;
    int bad = 0;
    for (int64_t j = 0; j < n; ++j) {
        if (owner_tl[j] < 0) { bad = 1; owner[j] = -1; continue; }
        owner[j] = (int32_t)midx[owner_tl[j]];
    }

    /* Step 4. Merged sequence m (Alg. 1 lines 10-17): tokens are the survivor's;
     * mask is the OR over members; log-prob / src come from the largest member index with mask 1
     * there (the inner loop visits j in descending order and only writes blocks not yet llm). */
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t m = 0; m < M; ++m) {
        int64_t s = merged_origin[m];
        int64_t Ls = offsets[s + 1] - offsets[s];
        int64_t base = merged_offsets[m];
        for (int64_t p = 0; p < Ls; ++p) {
            merged_tokens[base + p] = tokens[offsets[s] + p];
            merged_mask[base + p] = 0;
            merged_src[base + p] = -1;
            if (merged_old_logp) merged_old_logp[base + p] = 0.0f;
        }
        for (int64_t j = 0; j <= s; ++j) { /* members G_m = {j : owner_tl(j) = s}, includes s; ascending */
            if (owner_tl[j] != s) continue;
            int64_t Lj = offsets[j + 1] - offsets[j];
            for (int64_t p = 0; p < Lj; ++p) {
                if (!mask_at(resp_start, mask_in, offsets, j, p)) continue;
                merged_mask[base + p] = 1;            /* OR over members */
                merged_src[base + p] = (int32_t)j;    /* ascending j: the last writer is max K */
                if (merged_old_logp) merged_old_logp[base + p] = old_logp_in ? old_logp_in[offsets[j] + p] : 0.0f;
            }
        }
    }

    free(survives); free(last_ext); free(owner_tl); free(midx);
    return bad ? -2 : 0;
}

/* ------------------------------------------------------------------------------------------ loss */

static double load_logit(const void* logits, int dtype, int64_t idx) {
    if (dtype == 1) return (double)((const float*)logits)[idx];
    /* bf16: the upper 16 bits of an IEEE binary32; conversion to fp64 is exact */
    uint32_t bits = ((uint32_t)((const uint16_t*)logits)[idx]) << 16;
    float f;
    memcpy(&f, &bits, 4);
    return (double)f;
}

/*
 * Loss oracle (steps 1-7).  The paper gives no formula ("GRPO-style policy-gradient
 * updates" PAPER.md:91; clip_ratio = 0.2 PAPER.md:531); the definition is BASELINE.json north_star's
 * sentence: log-softmax, target gather, importance ratio vs old log-probs, PPO/GRPO clip, masked
 * per-trajectory mean, gradient w.r.t. logits.
 *
 * Per-token vectors cover ALL T tokens of the call (needed for the normalisers N_s, S').  The logits
 * matrix may be given for a subset of R rows only: row r of `logits` is token row_ids[r] (row_ids
 * NULL => R == T and row r is token r).  This lets full-size parity be checked on sampled rows and the
 * scalar be accumulated slab by slab.
 *
 * Outputs (all optional except loss_partial): loss_partial[1] = sum over the given rows of w_t L_t;
 * logp[R], w[R], g[R], Lt[R]; dlogits[R*V] (fp64, before any rounding);
 * stats[4] += {sum m_t, #clipped high, #clipped low, sum w_t (-log r_t)} over the given rows.
 * Returns 0; -1 invalid argument; -3 target or segment id out of range on a masked-in row.
 */
/*
 * Extended form (DESIGN.md "O-L" steps 8-9; the "other loss terms" of PAPER.md:136 that the protocol of PAPER.md:531 names:
 * kl_loss_coef = 2e-3 with the `low_var_kl` estimator, and the policy entropy the paper monitors):
 *   step 8  d_t = ref_logp_t - logp_t;  k3_t = min(exp(d_t) - d_t - 1, 10)   (the low-variance "k3" estimator of
 *           KL(pi || pi_ref), clamped at 10; reading L-16);  loss += kl_coef sum_t w_t k3_t;
 *           g_t += grad_scale w_t kl_coef (1 - exp(d_t)) [k3_t < 10]
 *   step 9  H_t = lse_t - sum_v p_tv z_tv  (entropy of the row's softmax; reported, no gradient)
 * ref_logp NULL or kl_coef 0 switches step 8 off.  k3[R], ent[R] optional; ext[2] += {sum w_t k3_t, sum w_t H_t}.
 *   step 3b (optional, clip_c > 0; reading L-18: the three-parameter "dual-clip" bound of SURVEY.md §8(f) f1): for A_t < 0
 *           the surrogate is capped, L_t = min(L_t, -A_t c); where the cap is strictly active (r_t > c) the gradient is zero.
 */
static int loss_impl(const void* logits, int32_t dtype, int64_t R, int32_t V, int64_t ld, const int64_t* row_ids,
                     const int32_t* targets, const float* old_logp, const float* adv, const uint8_t* mask,
                     const int32_t* seg_ids, int64_t T, int32_t S,
                     double eps_lo, double eps_hi, const float* seg_denom, double inv_num_segs, double grad_scale,
                     double* loss_partial, double* logp, double* w, double* g, double* Lt, double* dlogits,
                     double* stats, const float* ref_logp, double kl_coef, double* k3, double* ent, double* ext, double clip_c) {
    if (R < 0 || T < 0 || V <= 0 || S <= 0 || ld < V || eps_lo < 0 || eps_hi < 0 || clip_c < 0) return -1;
    if (dtype != 0 && dtype != 1) return -1;

    /* Step 4: N_s = sum_{t: s_t = s} m_t (or seg_denom[s]);  S' = #{s: N_s > 0} (or 1/inv_num_segs). */
    double* Ns = (double*)calloc((size_t)S, sizeof(double));
    int err = 0;
    for (int64_t t = 0; t < T; ++t) {
        if (!mask[t]) continue;
        if (seg_ids[t] < 0 || seg_ids[t] >= S) { err = -3; continue; }
        Ns[seg_ids[t]] += 1.0;
    }
    if (seg_denom)
        for (int32_t s = 0; s < S; ++s) Ns[s] = (double)seg_denom[s];
    double Sp = 0.0;
    for (int32_t s = 0; s < S; ++s) Sp += (Ns[s] > 0.0);
    double inv_Sp = (inv_num_segs != 0.0) ? inv_num_segs : (Sp > 0.0 ? 1.0 / Sp : 0.0);

    /* Per-row terms are stored and summed afterwards in row order, so the scalar does not depend on the
     * number of threads (step 5 is a plain sum over t). */
    double* term = (double*)calloc((size_t)(R > 0 ? R : 1) * 7, sizeof(double)); /* {w L, m, clip_hi, clip_lo, w(-log r), w k3, w H} */
#pragma omp parallel for schedule(static) reduction(min : err)
    for (int64_t r = 0; r < R; ++r) {
        int64_t t = row_ids ? row_ids[r] : r;
        double* drow = dlogits ? dlogits + r * (int64_t)V : NULL;
        if (logp) logp[r] = 0.0;
        if (w) w[r] = 0.0;
        if (g) g[r] = 0.0;
        if (Lt) Lt[r] = 0.0;
        if (k3) k3[r] = 0.0;
        if (ent) ent[r] = 0.0;
        if (drow) for (int32_t v = 0; v < V; ++v) drow[v] = 0.0;
        if (t < 0 || t >= T) { err = -1; continue; }
        if (!mask[t]) continue; /* m_t = 0: contributes nothing, dlogits row is zero (L-14) */
        int32_t y = targets[t], sg = seg_ids[t];
        if (y < 0 || y >= V || sg < 0 || sg >= S) { err = -3; continue; }
        const int64_t base = r * ld;

        /* Step 1: lse = max + log sum exp(z - max); logp = z_y - lse; p_v = exp(z_v - lse). */
        double zmax = load_logit(logits, dtype, base);
        for (int32_t v = 1; v < V; ++v) {
            double z = load_logit(logits, dtype, base + v);
            if (z > zmax) zmax = z;
        }
        double sum = 0.0;
        for (int32_t v = 0; v < V; ++v) sum += exp(load_logit(logits, dtype, base + v) - zmax);
        double lse = zmax + log(sum);
        double lp = load_logit(logits, dtype, base + y) - lse;

        /* Step 2: r = exp(logp - old_logp). */
        double ratio = exp(lp - (double)old_logp[t]);
        double A = (double)adv[t];

        /* Step 3: L = -min(r A, clip(r, 1-eps_lo, 1+eps_hi) A). */
        double rc = ratio;
        if (rc < 1.0 - eps_lo) rc = 1.0 - eps_lo;
        if (rc > 1.0 + eps_hi) rc = 1.0 + eps_hi;
        double a1 = ratio * A, a2 = rc * A;
        double L = -(a1 < a2 ? a1 : a2);

        /* Step 3b: dual-clip cap for negative advantages, L = min(L, -A c). */
        int cap = 0;
        if (clip_c > 0.0 && A < 0.0) {
            double L3 = -A * clip_c;
            if (L3 < L) { L = L3; cap = 1; }
        }

        /* Step 4: w = m / (N_s S'). */
        double wt = (Ns[sg] > 0.0) ? inv_Sp / Ns[sg] : 0.0;

        /* Step 6: pass = not(A>0 and r>1+eps_hi) and not(A<0 and r<1-eps_lo);
         * g = grad_scale w (-A r) [pass]; dlogits_v = g (1[v=y] - p_v). */
        int clip_hi = (A > 0.0 && ratio > 1.0 + eps_hi);
        int clip_lo = (A < 0.0 && ratio < 1.0 - eps_lo);
        double gt = (clip_hi || clip_lo || cap) ? 0.0 : grad_scale * wt * (-A * ratio);

        /* Step 8: low-variance KL estimator against the reference policy's log-prob of the same token. */
        double k3t = 0.0;
        if (ref_logp && kl_coef != 0.0) {
            double d = (double)ref_logp[t] - lp;
            k3t = exp(d) - d - 1.0;
            if (k3t < 10.0) gt += grad_scale * wt * kl_coef * (1.0 - exp(d));
            else k3t = 10.0;
        }

        /* Step 9: entropy of the row, H = lse - sum_v p_v z_v. */
        double pz = 0.0;
        for (int32_t v = 0; v < V; ++v) {
            double z = load_logit(logits, dtype, base + v);
            pz += exp(z - lse) * z;
        }
        double H = lse - pz;
        term[7 * r + 5] = wt * k3t;
        term[7 * r + 6] = wt * H;
        if (k3) k3[r] = k3t;
        if (ent) ent[r] = H;

        term[7 * r + 0] = wt * L; /* step 5 */
        term[7 * r + 1] = 1.0; term[7 * r + 2] = clip_hi; term[7 * r + 3] = clip_lo;
        term[7 * r + 4] = wt * (-(lp - (double)old_logp[t]));
        if (logp) logp[r] = lp;
        if (w) w[r] = wt;
        if (g) g[r] = gt;
        if (Lt) Lt[r] = L;
        if (drow) {
            for (int32_t v = 0; v < V; ++v) {
                double p = exp(load_logit(logits, dtype, base + v) - lse);
                drow[v] = gt * ((v == y ? 1.0 : 0.0) - p);
            }
        }
    }
    double total = 0.0, st0 = 0, st1 = 0, st2 = 0, st3 = 0, kl = 0, en = 0;
    for (int64_t r = 0; r < R; ++r) {
        total += term[7 * r + 0];
        st0 += term[7 * r + 1]; st1 += term[7 * r + 2]; st2 += term[7 * r + 3]; st3 += term[7 * r + 4];
        kl += term[7 * r + 5]; en += term[7 * r + 6];
    }
    *loss_partial = total + kl_coef * kl;   /* step 5 (+ step 8) */
    if (stats) { stats[0] += st0; stats[1] += st1; stats[2] += st2; stats[3] += st3; }
    if (ext) { ext[0] += kl; ext[1] += en; }
    free(term);
    free(Ns);
    return err;
}

int ajt_oracle_loss(const void* logits, int32_t dtype, int64_t R, int32_t V, int64_t ld, const int64_t* row_ids,
                    const int32_t* targets, const float* old_logp, const float* adv, const uint8_t* mask,
                    const int32_t* seg_ids, int64_t T, int32_t S,
                    double eps_lo, double eps_hi, const float* seg_denom, double inv_num_segs, double grad_scale,
                    double* loss_partial, double* logp, double* w, double* g, double* Lt, double* dlogits,
                    double* stats) {
    return loss_impl(logits, dtype, R, V, ld, row_ids, targets, old_logp, adv, mask, seg_ids, T, S, eps_lo, eps_hi, seg_denom,
                     inv_num_segs, grad_scale, loss_partial, logp, w, g, Lt, dlogits, stats, NULL, 0.0, NULL, NULL, NULL, 0.0);
}

int ajt_oracle_loss_ex(const void* logits, int32_t dtype, int64_t R, int32_t V, int64_t ld, const int64_t* row_ids,
                       const int32_t* targets, const float* old_logp, const float* adv, const uint8_t* mask,
                       const int32_t* seg_ids, int64_t T, int32_t S,
                       double eps_lo, double eps_hi, const float* seg_denom, double inv_num_segs, double grad_scale,
                       double* loss_partial, double* logp, double* w, double* g, double* Lt, double* dlogits,
                       double* stats, const float* ref_logp, double kl_coef, double* k3, double* ent, double* ext) {
    return loss_impl(logits, dtype, R, V, ld, row_ids, targets, old_logp, adv, mask, seg_ids, T, S, eps_lo, eps_hi, seg_denom,
                     inv_num_segs, grad_scale, loss_partial, logp, w, g, Lt, dlogits, stats, ref_logp, kl_coef, k3, ent, ext, 0.0);
}

int ajt_oracle_loss_ex2(const void* logits, int32_t dtype, int64_t R, int32_t V, int64_t ld, const int64_t* row_ids,
                        const int32_t* targets, const float* old_logp, const float* adv, const uint8_t* mask,
                        const int32_t* seg_ids, int64_t T, int32_t S,
                        double eps_lo, double eps_hi, const float* seg_denom, double inv_num_segs, double grad_scale,
                        double* loss_partial, double* logp, double* w, double* g, double* Lt, double* dlogits,
                        double* stats, const float* ref_logp, double kl_coef, double* k3, double* ent, double* ext, double clip_c) {
    return loss_impl(logits, dtype, R, V, ld, row_ids, targets, old_logp, adv, mask, seg_ids, T, S, eps_lo, eps_hi, seg_denom,
                     inv_num_segs, grad_scale, loss_partial, logp, w, g, Lt, dlogits, stats, ref_logp, kl_coef, k3, ent, ext, clip_c);
}

/* Round an fp64 value to bf16 (round-to-nearest-even), returned as fp64 (reading L-10:
 * the oracle rounds its fp64 value to bf16 directly). bf16 = 8 exponent bits, 7 stored mantissa bits. */
double ajt_oracle_round_bf16(double x) {
    if (x == 0.0 || !isfinite(x)) return x;
    int e;
    double m = frexp(x, &e);          /* x = m 2^e, 0.5 <= |m| < 1 */
    int emin = -126;                  /* smallest normal exponent of binary32/bf16 (value 2^-126) */
    int ulp_exp = e - 8;              /* 8 significant bits: ulp = 2^(e-8) */
    if (e - 1 < emin) ulp_exp = emin - 7; /* subnormal range: fixed ulp 2^-133 */
    (void)m;
    double scaled = ldexp(x, -ulp_exp);
    double rn = nearbyint(scaled);    /* default rounding mode: to nearest, ties to even */
    return ldexp(rn, ulp_exp);
}

int ajt_oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void ajt_oracle_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

void ajt_oracle_round_bf16_array(const double* in, double* out, int64_t n) {
    for (int64_t i = 0; i < n; ++i) out[i] = ajt_oracle_round_bf16(in[i]);
}

/* ------------------------------------------------------------------------------ block-level merge */

#define ORACLE_AUTHOR_LLM 2   /* author labels: 0 env, 1 user, 2 llm (eq. (1)) */
#define ORACLE_MATCH_TEXT 0   /* "text (default): exact text match at every aligned position" */
#define ORACLE_MATCH_TOKEN 1  /* "token: exact token-id match at every aligned position" */

/* Match(S^[k], T^[k]) of PAPER.md:182 for block sb of S and block tb of T.  The text m of a block is represented by a
 * caller-supplied 64-bit id with id equality <=> text equality (reading B-1). */
static int block_match(const int64_t* block_ids, const int64_t* tok_off, const int32_t* tokens, int64_t sb, int64_t tb,
                       int32_t match_mode) {
    if (match_mode == ORACLE_MATCH_TEXT) return block_ids[sb] == block_ids[tb];
    int64_t ls = tok_off[sb + 1] - tok_off[sb], lt = tok_off[tb + 1] - tok_off[tb];
    if (ls != lt) return 0;
    for (int64_t p = 0; p < ls; ++p)
        if (tokens[tok_off[sb] + p] != tokens[tok_off[tb] + p]) return 0;
    return 1;
}

/*
 * Block-level timeline merging: Algorithm 1 followed line by line on timelines of
 * message blocks (eq. (1)), per episode (timelines with different traj_ids are never compared, M-4).
 *
 * Timeline i = blocks block_offsets[i] .. block_offsets[i+1]; block b = (text id block_ids[b], author[b], tokens /
 * logp / tok_mask at tok_off[b] .. tok_off[b+1]).  tok_mask NULL => mu = 1 exactly on the tokens of llm blocks
 * (PAPER.md:176).  logp may be NULL.
 *
 * Outputs (caller-allocated at worst-case capacity: all tokens, all blocks, n sequences):
 *   merged_tokens / merged_mask / merged_logp / merged_tok_src [N_out]  (tok_src = timeline whose block supplied the token
 *   where the mask is 1, else -1), merged_offsets[M+1] (tokens), merged_block_offsets[M+1] (blocks),
 *   merged_block_src[B_out] (timeline whose block k stands at block k of the survivor), merged_block_author[B_out],
 *   merged_block_tok_off[B_out+1], merged_origin[M], merged_traj[M], owner[n], counts[3] = {M, B_out, N_out}.
 * Returns 0, or -1 on invalid input.
 */
int ajt_oracle_merge_blocks(const int64_t* block_ids, const int64_t* block_offsets, const int32_t* traj_ids,
                            const uint8_t* author, const int64_t* tok_off, const int32_t* tokens, const float* logp,
                            const uint8_t* tok_mask, int32_t n, int32_t match_mode,
                            int32_t* merged_tokens, uint8_t* merged_mask, float* merged_logp, int32_t* merged_tok_src,
                            int64_t* merged_offsets, int64_t* merged_block_offsets, int32_t* merged_block_src,
                            uint8_t* merged_block_author, int64_t* merged_block_tok_off,
                            int32_t* merged_origin, int32_t* merged_traj, int32_t* owner, int64_t* counts) {
    if (n < 0 || (match_mode != ORACLE_MATCH_TEXT && match_mode != ORACLE_MATCH_TOKEN)) return -1;
    if (block_offsets[0] != 0) return -1;
    for (int64_t i = 0; i < n; ++i)
        if (block_offsets[i + 1] - block_offsets[i] < 1) return -1;   /* K_i >= 1 */
    const int64_t B = block_offsets[n];
    if (tok_off[0] != 0) return -1;
    for (int64_t b = 0; b < B; ++b)
        if (tok_off[b + 1] < tok_off[b]) return -1;

    /* the mutable part of every block: author and where its tokens / logprobs come from (Alg. 1 lines 12-14) */
    uint8_t* cur_author = (uint8_t*)malloc((size_t)B + 1);
    int32_t* cur_src = (int32_t*)malloc(sizeof(int32_t) * ((size_t)B + 1));
    uint8_t* absorbed = (uint8_t*)calloc((size_t)n + 1, 1);            /* the set A, line 1 */
    int64_t* absorber = (int64_t*)malloc(sizeof(int64_t) * ((size_t)n + 1));
    for (int64_t i = 0; i < n; ++i) {
        absorber[i] = i;
        for (int64_t b = block_offsets[i]; b < block_offsets[i + 1]; ++b) { cur_author[b] = author[b]; cur_src[b] = (int32_t)i; }
    }

    for (int64_t i = n - 1; i >= 1; --i) {                               /* line 2 */
        if (absorbed[i]) continue;                                       /* lines 3-5 */
        const int64_t Ki = block_offsets[i + 1] - block_offsets[i];
        for (int64_t j = i - 1; j >= 0; --j) {                           /* line 6 */
            if (absorbed[j]) continue;                                   /* lines 7-8 */
            if (traj_ids[j] != traj_ids[i]) continue;                    /* one list per episode (M-4) */
            const int64_t Kj = block_offsets[j + 1] - block_offsets[j];
            if (Ki < Kj) continue;                                       /* line 9: |T_i| >= |T_j| */
            int ok = 1;
            for (int64_t k = 0; k < Kj && ok; ++k)                       /* line 9: Match for all k in [1, |T_j|] */
                ok = block_match(block_ids, tok_off, tokens, block_offsets[i] + k, block_offsets[j] + k, match_mode);
            if (!ok) continue;
            for (int64_t k = 0; k < Kj; ++k) {                           /* line 10 */
                const int64_t bi = block_offsets[i] + k, bj = block_offsets[j] + k;
                if (cur_author[bj] == ORACLE_AUTHOR_LLM && cur_author[bi] != ORACLE_AUTHOR_LLM) {   /* line 11 */
                    cur_author[bi] = ORACLE_AUTHOR_LLM;                  /* line 12 */
                    cur_src[bi] = cur_src[bj];                           /* lines 13-14: tokens and logprob of T_j^[k] */
                }
            }
            absorbed[j] = 1;                                             /* line 18 */
            absorber[j] = i;
        }
    }

    /* line 22: survivors in original order, flattened */
    int64_t M = 0, Bout = 0, Nout = 0;
    int64_t* midx = (int64_t*)malloc(sizeof(int64_t) * ((size_t)n + 1));
    for (int64_t s = 0; s < n; ++s) {
        midx[s] = -1;
        if (absorbed[s]) continue;
        midx[s] = M;
        merged_origin[M] = (int32_t)s;
        merged_traj[M] = traj_ids[s];
        merged_offsets[M] = Nout;
        merged_block_offsets[M] = Bout;
        const int64_t Ks = block_offsets[s + 1] - block_offsets[s];
        for (int64_t k = 0; k < Ks; ++k) {
            const int64_t b = block_offsets[s] + k;
            const int64_t sj = cur_src[b];
            const int64_t sb = block_offsets[sj] + k;                    /* block k of the supplying timeline */
            merged_block_src[Bout] = (int32_t)sj;
            merged_block_author[Bout] = cur_author[b];
            merged_block_tok_off[Bout] = Nout;
            for (int64_t q = tok_off[sb]; q < tok_off[sb + 1]; ++q) {
                const int mk = tok_mask ? (tok_mask[q] != 0) : (cur_author[b] == ORACLE_AUTHOR_LLM);
                merged_tokens[Nout] = tokens[q];
                merged_mask[Nout] = (uint8_t)mk;
                merged_tok_src[Nout] = mk ? (int32_t)sj : -1;
                if (merged_logp) merged_logp[Nout] = (logp && mk) ? logp[q] : 0.0f;
                ++Nout;
            }
            ++Bout;
        }
        ++M;
    }
    merged_offsets[M] = Nout;
    merged_block_offsets[M] = Bout;
    merged_block_tok_off[Bout] = Nout;
    for (int64_t j = 0; j < n; ++j) owner[j] = (int32_t)midx[absorber[j]];
    counts[0] = M; counts[1] = Bout; counts[2] = Nout;
    free(cur_author); free(cur_src); free(absorbed); free(absorber); free(midx);
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * Per-token loss inputs from merged sequences (reading L-12), sequence by sequence: inside sequence m the
 * row at position q predicts the token at q + 1, so targets / mask / old_logp are those of q + 1; the last position of
 * every sequence has nothing to predict (0, 0, 0).  seg_ids = dense trajectory id of the surviving timeline; adv = that
 * trajectory's advantage.  merged_old_logp / old_logp and seg_adv / adv may be NULL in pairs.  The same loops as the
 * Python function oracle.pack_loss_inputs had (its pins, tests/test_oracle_pack.py, run against this one). */
int ajt_oracle_pack(const int32_t* merged_tokens, const uint8_t* merged_mask, const float* merged_old_logp,
                    const int64_t* merged_offsets, const int32_t* merged_origin, const int32_t* tl_seg, const float* seg_adv,
                    int64_t M, int32_t* targets, uint8_t* mask, float* old_logp, int32_t* seg_ids, float* adv) {
    for (int64_t m = 0; m < M; ++m) {
        const int64_t a = merged_offsets[m], b = merged_offsets[m + 1];
        if (b < a) return -1;
        const int32_t sg = tl_seg[merged_origin[m]];
        for (int64_t q = a; q < b; ++q) {
            seg_ids[q] = sg;
            if (adv) adv[q] = seg_adv[sg];
            if (q + 1 < b) {
                targets[q] = merged_tokens[q + 1];
                mask[q] = merged_mask[q + 1] ? 1 : 0;
                if (old_logp) old_logp[q] = merged_old_logp[q + 1];
            } else {
                targets[q] = 0;
                mask[q] = 0;
                if (old_logp) old_logp[q] = 0.0f;
            }
        }
    }
    return 0;
}
