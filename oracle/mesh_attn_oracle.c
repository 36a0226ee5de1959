/*
 * mesh_attn_oracle.c -- TEST INFRASTRUCTURE ONLY. Not part of the product path.
 *
 * Plain, slow, fp64 CPU oracle for what the Mesh-Attention per-GPU compute core
 * must produce.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference leg may call it.  It shares no code with the CUDA path.
 *
 * The method reaches *exactly* full softmax attention ("merged
 * exactly", L188 "the exact attention output of Q_g over all KV partitions"), so
 * the oracle is the definition written out:
 *
 *      O = softmax(Q K^T / sqrt(d)) V
 *
 * evaluated in double precision on the bf16 input bits widened to double, with
 *   - causal masking "each token can attend only to itself and preceding tokens"
 *      decided on explicit token positions pos[row] handed in by
 *     the caller (the oracle never calls the planner);
 *   - GQA: "each group of g consecutive query heads share one KV head"
 *     (PAPER.md L427): query head h reads KV head h / (Hq/Hkv);
 *   - LSE = natural log of the sum of exp of the *scaled* scores, one scalar per
 *     (query position, head) (reading R2);
 *   - a row with no visible key has O = 0 and LSE = -inf (reading R5).
 *
 * Backward is the derivative of that definition with upstream dO (PAPER.md
 * L234-236 names the inputs Q, KV, O, dO; reading R8):
 *      P  = exp(S - LSE)            dV[t] = sum_s P[s,t] dO[s]
 *      dP[s,t] = dO[s] . v[t]       Delta[s] = dO[s] . O[s]
 *      dS = P o (dP - Delta)        dQ[s] = scale sum_t dS[s,t] k[t]
 *                                   dK[t] = scale sum_s dS[s,t] q[s]
 * with dK, dV summed over the g query heads of a GQA group.
 *
 * Tensor layout: [N rows][H heads][D] bf16 (uint16 bit patterns), one batch
 * element per call.  No blocking, no fusion, no online softmax: two passes per
 * row (max, then sum), exactly as the definition reads.
 *
 * Pins (tests/test_oracle_pins.py): brute-force triple loops, closed forms
 * (uniform keys -> mean of V, dominant key -> that V row, key shift invariance),
 * merge of any tiling == full attention, finite differences, global gradient
 * invariants, torch CPU fp64 softmax+autograd as a library second opinion.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static inline double bf16_to_f64(uint16_t b)
{
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* element (row, h, d) of a [N][H][D] tensor */
#define AT(T, H, D, row, h, d) ((T)[((size_t)(row) * (size_t)(H) + (size_t)(h)) * (size_t)(D) + (size_t)(d)])

/* visible(s, t): non-causal -> always; causal -> pos[t] <= pos[s].
 * key_sel (may be NULL) restricts the key set: used for the per-pair partial
 * Attention(Q_i, K_j, V_j) of PAPER.md L81-84. */
static inline int visible(int causal, const int64_t *pos, const uint8_t *key_sel, int64_t s, int64_t t)
{
    if (key_sel && !key_sel[t]) return 0;
    if (causal && pos[t] > pos[s]) return 0;
    return 1;
}

/* scaled score S[s,t] = scale * sum_d q[s,d] k[t,d] */
static inline double score(const uint16_t *Q, const uint16_t *K, int Hq, int Hkv, int D,
                           int64_t s, int h, int hk, int64_t t, double scale)
{
    double acc = 0.0;
    for (int d = 0; d < D; ++d)
        acc += bf16_to_f64(AT(Q, Hq, D, s, h, d)) * bf16_to_f64(AT(K, Hkv, D, t, hk, d));
    return scale * acc;
}

/*
 * Forward rows.  For sample k: query row qrows[k], query head qheads[k].
 *   O_out[k*D + d], lse_out[k].
 * Definition, two passes: m = max_t S; l = sum_t exp(S - m); LSE = m + ln l;
 * O = sum_t exp(S - LSE) v[t].
 */
void oracle_attn_fwd_rows(const uint16_t *Q, const uint16_t *K, const uint16_t *V,
                          int64_t N, int Hq, int Hkv, int D, double scale, int causal,
                          const int64_t *pos, const uint8_t *key_sel,
                          int64_t nq, const int64_t *qrows, const int32_t *qheads,
                          double *O_out, double *lse_out)
{
    const int g = Hq / Hkv;
#pragma omp parallel
    {
        double *S = (double *)malloc((size_t)N * sizeof(double));
#pragma omp for schedule(dynamic, 1)
        for (int64_t k = 0; k < nq; ++k) {
            const int64_t s = qrows[k];
            const int h = qheads[k], hk = h / g;
            double m = -INFINITY;
            for (int64_t t = 0; t < N; ++t) {
                if (!visible(causal, pos, key_sel, s, t)) { S[t] = -INFINITY; continue; }
                S[t] = score(Q, K, Hq, Hkv, D, s, h, hk, t, scale);
                if (S[t] > m) m = S[t];
            }
            double *o = O_out + (size_t)k * D;
            for (int d = 0; d < D; ++d) o[d] = 0.0;
            if (m == -INFINITY) { lse_out[k] = -INFINITY; continue; } /* no visible key */
            double l = 0.0;
            for (int64_t t = 0; t < N; ++t)
                if (S[t] != -INFINITY) l += exp(S[t] - m);
            const double lse = m + log(l);
            lse_out[k] = lse;
            for (int64_t t = 0; t < N; ++t) {
                if (S[t] == -INFINITY) continue;
                const double p = exp(S[t] - lse);
                for (int d = 0; d < D; ++d) o[d] += p * bf16_to_f64(AT(V, Hkv, D, t, hk, d));
            }
        }
        free(S);
    }
}

/*
 * Online-softmax reducer as a plain formula (formula not
 * printed, reading R4): for m partials (O_k, lse_k) of one (row, head)
 *     lse* = ln sum_k exp(lse_k),   O = sum_k exp(lse_k - lse*) O_k
 * evaluated with max subtraction; a partial with lse_k = -inf has weight 0; all
 * -inf gives (0, -inf).
 */
void oracle_attn_merge(int m, int D, const double *O_parts, const double *lse_parts,
                       double *O_out, double *lse_out)
{
    double mx = -INFINITY;
    for (int k = 0; k < m; ++k) if (lse_parts[k] > mx) mx = lse_parts[k];
    for (int d = 0; d < D; ++d) O_out[d] = 0.0;
    if (mx == -INFINITY) { *lse_out = -INFINITY; return; }
    double sum = 0.0;
    for (int k = 0; k < m; ++k) if (lse_parts[k] != -INFINITY) sum += exp(lse_parts[k] - mx);
    const double lse = mx + log(sum);
    *lse_out = lse;
    for (int k = 0; k < m; ++k) {
        if (lse_parts[k] == -INFINITY) continue;
        const double w = exp(lse_parts[k] - lse);
        for (int d = 0; d < D; ++d) O_out[d] += w * O_parts[(size_t)k * D + d];
    }
}

/*
 * Backward, query side.  For sample k (row s, head h):
 *   recompute S, LSE, O from the definition; Delta = dO[s].O[s];
 *   dQ[s] = scale * sum_t P[s,t] (dO[s].v[t] - Delta) k[t].
 * Also returns lse_out[k], delta_out[k] (may be NULL).
 */
void oracle_attn_bwd_dq_rows(const uint16_t *Q, const uint16_t *K, const uint16_t *V, const uint16_t *dO,
                             int64_t N, int Hq, int Hkv, int D, double scale, int causal,
                             const int64_t *pos,
                             int64_t nq, const int64_t *qrows, const int32_t *qheads,
                             double *dQ_out, double *lse_out, double *delta_out)
{
    const int g = Hq / Hkv;
#pragma omp parallel
    {
        double *S = (double *)malloc((size_t)N * sizeof(double));
        double *o = (double *)malloc((size_t)D * sizeof(double));
#pragma omp for schedule(dynamic, 1)
        for (int64_t k = 0; k < nq; ++k) {
            const int64_t s = qrows[k];
            const int h = qheads[k], hk = h / g;
            double *dq = dQ_out + (size_t)k * D;
            for (int d = 0; d < D; ++d) { dq[d] = 0.0; o[d] = 0.0; }
            double m = -INFINITY;
            for (int64_t t = 0; t < N; ++t) {
                if (!visible(causal, pos, NULL, s, t)) { S[t] = -INFINITY; continue; }
                S[t] = score(Q, K, Hq, Hkv, D, s, h, hk, t, scale);
                if (S[t] > m) m = S[t];
            }
            if (m == -INFINITY) {
                if (lse_out) lse_out[k] = -INFINITY;
                if (delta_out) delta_out[k] = 0.0;
                continue;
            }
            double l = 0.0;
            for (int64_t t = 0; t < N; ++t) if (S[t] != -INFINITY) l += exp(S[t] - m);
            const double lse = m + log(l);
            for (int64_t t = 0; t < N; ++t) {
                if (S[t] == -INFINITY) continue;
                const double p = exp(S[t] - lse);
                for (int d = 0; d < D; ++d) o[d] += p * bf16_to_f64(AT(V, Hkv, D, t, hk, d));
            }
            double delta = 0.0;
            for (int d = 0; d < D; ++d) delta += bf16_to_f64(AT(dO, Hq, D, s, h, d)) * o[d];
            for (int64_t t = 0; t < N; ++t) {
                if (S[t] == -INFINITY) continue;
                const double p = exp(S[t] - lse);
                double dp = 0.0;
                for (int d = 0; d < D; ++d)
                    dp += bf16_to_f64(AT(dO, Hq, D, s, h, d)) * bf16_to_f64(AT(V, Hkv, D, t, hk, d));
                const double ds = p * (dp - delta);
                for (int d = 0; d < D; ++d) dq[d] += scale * ds * bf16_to_f64(AT(K, Hkv, D, t, hk, d));
            }
            if (lse_out) lse_out[k] = lse;
            if (delta_out) delta_out[k] = delta;
        }
        free(S);
        free(o);
    }
}

/*
 * Backward, key side.  For sample k (key row t, KV head hk):
 *   dV[t] = sum_{h in group(hk)} sum_{s in qs} P[s,t] dO[s]
 *   dK[t] = scale sum_{h in group(hk)} sum_{s in qs} P[s,t] (dO[s].v[t] - Delta[h,s]) q[s]
 * where qs = qs_rows[0..nqs) is the set of query rows summed over (all rows for
 * the true gradient; the rows with non-zero dO for the sparse-dO probe), and
 * lse_all / delta_all are [Hq][N] doubles holding LSE and Delta of those rows
 * (from oracle_attn_bwd_dq_rows).
 */
void oracle_attn_bwd_dkv_keys(const uint16_t *Q, const uint16_t *K, const uint16_t *V, const uint16_t *dO,
                              int64_t N, int Hq, int Hkv, int D, double scale, int causal,
                              const int64_t *pos,
                              int64_t nqs, const int64_t *qs_rows,
                              const double *lse_all, const double *delta_all,
                              int64_t nk, const int64_t *krows, const int32_t *kheads,
                              double *dK_out, double *dV_out)
{
    const int g = Hq / Hkv;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t k = 0; k < nk; ++k) {
        const int64_t t = krows[k];
        const int hk = kheads[k];
        double *dk = dK_out + (size_t)k * D;
        double *dv = dV_out + (size_t)k * D;
        for (int d = 0; d < D; ++d) { dk[d] = 0.0; dv[d] = 0.0; }
        for (int h = hk * g; h < (hk + 1) * g; ++h) {
            for (int64_t i = 0; i < nqs; ++i) {
                const int64_t s = qs_rows[i];
                if (!visible(causal, pos, NULL, s, t)) continue;
                const double lse = lse_all[(size_t)h * N + s];
                if (lse == -INFINITY) continue;
                const double p = exp(score(Q, K, Hq, Hkv, D, s, h, hk, t, scale) - lse);
                double dp = 0.0;
                for (int d = 0; d < D; ++d)
                    dp += bf16_to_f64(AT(dO, Hq, D, s, h, d)) * bf16_to_f64(AT(V, Hkv, D, t, hk, d));
                const double ds = p * (dp - delta_all[(size_t)h * N + s]);
                for (int d = 0; d < D; ++d) {
                    dv[d] += p * bf16_to_f64(AT(dO, Hq, D, s, h, d));
                    dk[d] += scale * ds * bf16_to_f64(AT(Q, Hq, D, s, h, d));
                }
            }
        }
    }
}
