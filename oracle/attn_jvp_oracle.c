/*
 * attn_jvp_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU statement of what the attention-JVP hot path computes,
 * written from the paper's definitions (App. B, Eq. 42-44), NOT from
 * Algorithm 1: the mask row, the scores s, the probabilities p and the score
 * tangents ts are materialised explicitly for every query row; there is no
 * tiling, no online softmax, no range list, no fusion.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or helper with paper_2606_25473_b200/ (the CUDA path), and the
 * CUDA path never calls it.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): central finite differences
 * of O along the tangent, brute-force dense masked attention written
 * independently in numpy, torch.func.jvp / SDPA / logsumexp, closed forms,
 * invariants and pair counts; the backward (attn_jvp_oracle_bwd) is pinned by torch.autograd, finite differences of
 * <O, dO> and invariants (tests/test_oracle_bwd_pins.py); the lse tangent (attn_jvp_oracle_rows_tl) by finite differences of
 * lse, torch.func.jvp(logsumexp) and closed forms (test_oracle_pins.py "TL").  Every exported function below is pinned; none is
 * "parity unpinned".
 *
 * Definitions followed (PAPER.md line : item):
 *   842-844  Eq. 42  O = softmax(Q K^T / sqrt(d) + M) V,  M in {0,-inf}
 *   846-848  Eq. 43  tS = (tQ K^T + Q tK^T) / sqrt(d)
 *   851-854  masked entries: S = -inf, tS = 0 (the mask has no tangent)
 *   862-864  Eq. 44  tO_a = sum_b p_ab tV_b + sum_b p_ab (tS_ab - sum_c p_ac tS_ac) V_b
 *   945      L = m + log(l)  (log-sum-exp of the scaled, masked scores)
 *   870-876  r = sum_b e^{s_ab - m} tS_ab, so r / l = sum_b p_ab tS_ab = mu_a: the tangent of L along the input
 *            tangent (d/d eps of log sum exp(S + eps tS) = softmax-weighted mean of tS); output `tlse`
 *   175-180  Eq. 8 / teacher-forcing mask over the packed [clean | noisy] sequence
 *   882-886  generic mask = query groups with key-range lists
 * Readings where the paper is silent are DESIGN.md R1 (both S and tS carry the
 * scale), R4 (exact TF predicate), R6 (block index), R9 (row with no allowed
 * key: O = 0, tO = 0, lse = -inf).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { AJO_MASK_FULL = 0, AJO_MASK_BLOCK_CAUSAL = 1, AJO_MASK_TEACHER_FORCING = 2, AJO_MASK_RANGES = 3 };
enum { AJO_F32 = 0, AJO_F64 = 1 };

typedef struct {
    int32_t kind;
    int32_t block_len;       /* C: tokens per block (frame_len * chunk_frames)          */
    int32_t num_blocks;      /* n: blocks (per half for TEACHER_FORCING)                */
    int32_t first_block_len; /* C1: tokens in block 0; 0 means C                        */
    /* AJO_MASK_RANGES only: group g owns query rows
       [q_begin[g], q_end[g]) and may see keys in the union of
       [k_begin[r], k_end[r]) for r in [range_offset[g], range_offset[g+1]).  */
    int32_t num_groups;
    const int32_t *q_begin, *q_end, *range_offset, *k_begin, *k_end;
} ajo_mask;

/* Block index of token x inside one half: blocks have length C1, C, C, ... (R6). */
static int64_t ajo_block_of(const ajo_mask *m, int64_t x)
{
    int64_t c1 = m->first_block_len > 0 ? m->first_block_len : m->block_len;
    if (x < c1) return 0;
    return 1 + (x - c1) / m->block_len;
}

static int64_t ajo_half_len(const ajo_mask *m)
{
    int64_t c1 = m->first_block_len > 0 ? m->first_block_len : m->block_len;
    return c1 + (int64_t)(m->num_blocks - 1) * m->block_len;
}

/* May query token a attend to key token b?  The plain predicate (R4). */
int attn_jvp_oracle_allowed(const ajo_mask *m, int64_t a, int64_t b)
{
    switch (m->kind) {
    case AJO_MASK_FULL:
        return 1;
    case AJO_MASK_BLOCK_CAUSAL:
        /* block i attends blocks <= i */
        return ajo_block_of(m, b) <= ajo_block_of(m, a);
    case AJO_MASK_TEACHER_FORCING: {
        /* packed sequence [clean | noisy] (Eq. 8) */
        int64_t half = ajo_half_len(m);
        int a_clean = a < half, b_clean = b < half;
        if (a_clean) {
            /* clean block i -> clean blocks <= i; clean never sees noisy */
            if (!b_clean) return 0;
            return ajo_block_of(m, b) <= ajo_block_of(m, a);
        } else {
            int64_t i = ajo_block_of(m, a - half);
            /* noisy block i -> clean blocks < i, plus noisy block i itself */
            if (b_clean) return ajo_block_of(m, b) < i;
            return ajo_block_of(m, b - half) == i;
        }
    }
    case AJO_MASK_RANGES:
        for (int g = 0; g < m->num_groups; ++g) {
            if (a < m->q_begin[g] || a >= m->q_end[g]) continue;
            for (int r = m->range_offset[g]; r < m->range_offset[g + 1]; ++r)
                if (b >= m->k_begin[r] && b < m->k_end[r]) return 1;
        }
        return 0;
    default:
        return 0;
    }
}

/* Unmasked (query, key) pairs of one head, by counting the predicate. */
int64_t attn_jvp_oracle_count_pairs(const ajo_mask *m, int64_t nq, int64_t nk)
{
    int64_t total = 0;
#pragma omp parallel for schedule(static) reduction(+ : total)
    for (int64_t a = 0; a < nq; ++a) {
        int64_t c = 0;
        for (int64_t b = 0; b < nk; ++b) c += attn_jvp_oracle_allowed(m, a, b);
        total += c;
    }
    return total;
}

static inline double ajo_load(const void *p, int dtype, int64_t idx)
{
    return dtype == AJO_F64 ? ((const double *)p)[idx] : (double)((const float *)p)[idx];
}

/*
 * One (batch, head) slice.  q, tq: [nq, d]; k, v, tk, tv: [nk, d]; rows contiguous
 * with stride d; dtype says whether they hold float or double (values are widened
 * exactly).  rows[0..nrows) lists the query rows to evaluate (NULL = rows 0..nrows-1).
 * Outputs, all fp64: o, to: [nrows, d]; lse: [nrows]; tlse: [nrows] or NULL (the tangent of lse, mu_a = sum_b p_ab
 * tS_ab = the paper's r / l; 0 for a row with no allowed key).
 * Returns 0, or -1 on a bad argument / allocation failure.
 */
int attn_jvp_oracle_rows_tl(const ajo_mask *mask, int64_t nq, int64_t nk, int32_t d, double scale,
                            int32_t dtype, const void *q, const void *k, const void *v,
                            const void *tq, const void *tk, const void *tv,
                            const int64_t *rows, int64_t nrows,
                            double *o, double *to, double *lse, double *tlse)
{
    if (!mask || nq <= 0 || nk <= 0 || d <= 0 || nrows < 0) return -1;
    if (dtype != AJO_F32 && dtype != AJO_F64) return -1;
    int failed = 0;
#pragma omp parallel
    {
        double *s = (double *)malloc(sizeof(double) * (size_t)nk);   /* scores, then p */
        double *ts = (double *)malloc(sizeof(double) * (size_t)nk);  /* score tangents */
        unsigned char *ok = (unsigned char *)malloc((size_t)nk);     /* mask row       */
        double *qa = (double *)malloc(sizeof(double) * (size_t)d);
        double *tqa = (double *)malloc(sizeof(double) * (size_t)d);
        if (!s || !ts || !ok || !qa || !tqa) {
#pragma omp atomic write
            failed = 1;
        }
        /* every thread reaches the worksharing loop or none does: the flag is read after a barrier */
#pragma omp barrier
        if (!failed) {
#pragma omp for schedule(dynamic, 1)
            for (int64_t i = 0; i < nrows; ++i) {
                int64_t a = rows ? rows[i] : i;
                double *oa = o + i * d, *toa = to + i * d;
                for (int c = 0; c < d; ++c) { oa[c] = 0.0; toa[c] = 0.0; }
                if (tlse) tlse[i] = 0.0;
                if (a < 0 || a >= nq) { lse[i] = NAN; continue; }
                for (int c = 0; c < d; ++c) {
                    qa[c] = ajo_load(q, dtype, a * d + c);
                    tqa[c] = ajo_load(tq, dtype, a * d + c);
                }
                /* mask row, Eq. 42 scores, Eq. 43 score tangents */
                double m = -INFINITY;
                for (int64_t b = 0; b < nk; ++b) {
                    ok[b] = (unsigned char)attn_jvp_oracle_allowed(mask, a, b);
                    if (!ok[b]) { s[b] = -INFINITY; ts[b] = 0.0; continue; }
                    double qk = 0.0, tqk = 0.0, qtk = 0.0;
                    for (int c = 0; c < d; ++c) {
                        double kb = ajo_load(k, dtype, b * d + c);
                        double tkb = ajo_load(tk, dtype, b * d + c);
                        qk += qa[c] * kb;
                        tqk += tqa[c] * kb;
                        qtk += qa[c] * tkb;
                    }
                    s[b] = scale * qk;
                    ts[b] = scale * (tqk + qtk);
                    if (s[b] > m) m = s[b];
                }
                if (m == -INFINITY) { lse[i] = -INFINITY; continue; } /* R9 */
                /* masked softmax over the allowed keys */
                double z = 0.0;
                for (int64_t b = 0; b < nk; ++b) {
                    s[b] = ok[b] ? exp(s[b] - m) : 0.0;
                    z += s[b];
                }
                for (int64_t b = 0; b < nk; ++b) s[b] /= z; /* s now holds p_ab */
                lse[i] = m + log(z);
                /* mu = sum_c p_ac tS_ac */
                double mu = 0.0;
                for (int64_t b = 0; b < nk; ++b) mu += s[b] * ts[b];
                if (tlse) tlse[i] = mu;
                /* O = sum p v;  Eq. 44 */
                for (int64_t b = 0; b < nk; ++b) {
                    if (!ok[b]) continue;
                    double p = s[b], w = p * (ts[b] - mu);
                    for (int c = 0; c < d; ++c) {
                        double vb = ajo_load(v, dtype, b * d + c);
                        double tvb = ajo_load(tv, dtype, b * d + c);
                        oa[c] += p * vb;
                        toa[c] += p * tvb + w * vb;
                    }
                }
            }
        }
        free(s); free(ts); free(ok); free(qa); free(tqa);
    }
    return failed ? -1 : 0;
}

/* The same without the lse tangent (the original entry point). */
int attn_jvp_oracle_rows(const ajo_mask *mask, int64_t nq, int64_t nk, int32_t d, double scale,
                         int32_t dtype, const void *q, const void *k, const void *v,
                         const void *tq, const void *tk, const void *tv,
                         const int64_t *rows, int64_t nrows,
                         double *o, double *to, double *lse)
{
    return attn_jvp_oracle_rows_tl(mask, nq, nk, d, scale, dtype, q, k, v, tq, tk, tv, rows, nrows, o, to, lse, NULL);
}

/*
 * Primal backward: the vector-Jacobian product of Eq. 42.  The paper gives no formula for it; it
 * only says the student's gradient flows through the ordinary primal path (Eq. 19) and that the forward
 * returns L for it.  This is the textbook VJP of O = softmax(S + M) V, S = scale * Q K^T, written out
 * with every row of P materialised:
 *     dV_b = sum_a p_ab dO_a
 *     dP_ab = <dO_a, v_b>,  delta_a = sum_b p_ab dP_ab,  dS_ab = p_ab (dP_ab - delta_a)     (softmax Jacobian)
 *     dQ_a = scale * sum_b dS_ab k_b,   dK_b = scale * sum_a dS_ab q_a
 * over the allowed pairs only (masked entries have p = 0 and the mask has no gradient).  Rows with no allowed key
 * contribute nothing and get dQ = 0.
 * Pass 1 runs over query rows (p row materialised; dQ, and lse_a, delta_a kept), pass 2 over keys (dK, dV), each
 * parallel over its own outputs so that no two threads add into the same element.
 * q, dout: [nq, d]; k, v: [nk, d].  rows / keys list the query rows / keys whose gradients are wanted (NULL = all);
 * dq: [nrows, d]; dk, dv: [nkeys, d], all fp64.  Pins: torch.autograd, finite differences of <O, dO>, invariants
 * (tests/test_oracle_bwd_pins.py).
 */
int attn_jvp_oracle_bwd(const ajo_mask *mask, int64_t nq, int64_t nk, int32_t d, double scale, int32_t dtype,
                        const void *q, const void *k, const void *v, const void *dout,
                        const int64_t *rows, int64_t nrows, const int64_t *keys, int64_t nkeys,
                        double *dq, double *dk, double *dv)
{
    if (!mask || nq <= 0 || nk <= 0 || d <= 0 || nrows < 0 || nkeys < 0) return -1;
    if (dtype != AJO_F32 && dtype != AJO_F64) return -1;
    double *lse = (double *)malloc(sizeof(double) * (size_t)nq);
    double *delta = (double *)malloc(sizeof(double) * (size_t)nq);
    int64_t *slot = (int64_t *)malloc(sizeof(int64_t) * (size_t)nq);   /* where row a's dQ goes, or -1 */
    if (!lse || !delta || !slot) { free(lse); free(delta); free(slot); return -1; }
    for (int64_t a = 0; a < nq; ++a) slot[a] = rows ? -1 : (a < nrows ? a : -1);
    if (rows) for (int64_t i = 0; i < nrows; ++i) if (rows[i] >= 0 && rows[i] < nq) slot[rows[i]] = i;
    for (int64_t i = 0; i < nrows * d; ++i) dq[i] = 0.0;
    int failed = 0;
#pragma omp parallel
    {
        double *p = (double *)malloc(sizeof(double) * (size_t)nk);    /* scores, then p_ab */
        double *dp = (double *)malloc(sizeof(double) * (size_t)nk);   /* dP_ab             */
        unsigned char *ok = (unsigned char *)malloc((size_t)nk);
        if (!p || !dp || !ok) {
#pragma omp atomic write
            failed = 1;
        }
#pragma omp barrier
        if (!failed) {
            /* pass 1: every query row (lse and delta of all rows are needed by pass 2) */
#pragma omp for schedule(dynamic, 1)
            for (int64_t a = 0; a < nq; ++a) {
                double m = -INFINITY;
                for (int64_t b = 0; b < nk; ++b) {
                    ok[b] = (unsigned char)attn_jvp_oracle_allowed(mask, a, b);
                    if (!ok[b]) { p[b] = -INFINITY; dp[b] = 0.0; continue; }
                    double qk = 0.0, dov = 0.0;
                    for (int c = 0; c < d; ++c) {
                        qk += ajo_load(q, dtype, a * d + c) * ajo_load(k, dtype, b * d + c);
                        dov += ajo_load(dout, dtype, a * d + c) * ajo_load(v, dtype, b * d + c);
                    }
                    p[b] = scale * qk;
                    dp[b] = dov;
                    if (p[b] > m) m = p[b];
                }
                if (m == -INFINITY) { lse[a] = -INFINITY; delta[a] = 0.0; continue; }
                double z = 0.0;
                for (int64_t b = 0; b < nk; ++b) { p[b] = ok[b] ? exp(p[b] - m) : 0.0; z += p[b]; }
                for (int64_t b = 0; b < nk; ++b) p[b] /= z;
                lse[a] = m + log(z);
                double dl = 0.0;
                for (int64_t b = 0; b < nk; ++b) dl += p[b] * dp[b];
                delta[a] = dl;
                if (slot[a] < 0) continue;
                double *dqa = dq + slot[a] * d;
                for (int64_t b = 0; b < nk; ++b) {
                    if (!ok[b]) continue;
                    double ds = p[b] * (dp[b] - dl);
                    for (int c = 0; c < d; ++c) dqa[c] += scale * ds * ajo_load(k, dtype, b * d + c);
                }
            }
            /* pass 2: the requested keys */
#pragma omp for schedule(dynamic, 1)
            for (int64_t j = 0; j < nkeys; ++j) {
                int64_t b = keys ? keys[j] : j;
                double *dkb = dk + j * d, *dvb = dv + j * d;
                for (int c = 0; c < d; ++c) { dkb[c] = 0.0; dvb[c] = 0.0; }
                if (b < 0 || b >= nk) continue;
                for (int64_t a = 0; a < nq; ++a) {
                    if (!attn_jvp_oracle_allowed(mask, a, b) || lse[a] == -INFINITY) continue;
                    double qk = 0.0, dov = 0.0;
                    for (int c = 0; c < d; ++c) {
                        qk += ajo_load(q, dtype, a * d + c) * ajo_load(k, dtype, b * d + c);
                        dov += ajo_load(dout, dtype, a * d + c) * ajo_load(v, dtype, b * d + c);
                    }
                    double pab = exp(scale * qk - lse[a]);
                    double ds = pab * (dov - delta[a]);
                    for (int c = 0; c < d; ++c) {
                        dvb[c] += pab * ajo_load(dout, dtype, a * d + c);
                        dkb[c] += scale * ds * ajo_load(q, dtype, a * d + c);
                    }
                }
            }
        }
        free(p); free(dp); free(ok);
    }
    free(lse); free(delta); free(slot);
    return failed ? -1 : 0;
}

/* Threads an oracle call will use (reported by bench.py as cpu_baseline.cores). */
int attn_jvp_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
