/*
 * jetlong_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU oracle for the Jet-Long bifocal RoPE attention hot path
 * (arxiv/paper_2607_07740).  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference leg may load this file.  It shares no code, header,
 * table or constant with the CUDA path under paper_2607_07740_b200/csrc/.
 *
 * Every function cites the passage of /root/reference/PAPER.md it follows ("P:nnn").
 * Readings of points the paper leaves open are the ones listed in DESIGN.md
 * ("Readings"), numbered R1..R16 after SURVEY.md section 8(c).
 *
 * Layouts (all contiguous, row-major):
 *   K, V   : [L, H_kv, d]  float32 (the exact bf16 / fp32 bit patterns the GPU gets,
 *                           widened; everything below is computed in double)
 *   Qrows  : [n, d]        float32, row j is Q[rows[j], heads[j], :]
 *   out    : [n, d]        double
 *   lse    : [n]           double   natural log of sum exp(scaled score)  (R8)
 *
 * Pins (tests/test_oracle_pins.py): Eq.(2) stepping incl. the printed 98304->3,
 * 98305->4; G=1 == causal control bit-exactly; three-call
 * inclusion-exclusion == direct masking; R_a R_b = R_{a+b};
 * closed-form cosine-sum scores for Eq.(1); Q=0 / constant-V softmax plumbing;
 * w0=0 and w0>=L-1 window edges; shift invariance; within-group aliasing
 * (P:220); brute force in pure Python on tiny inputs.
 * jlo_attend_rows_freq (frequency-interpolation map, a DEFINITION of this repository, R17): pinned by G=1 == causal,
 * gamma=1 == causal, gamma=0 == brute-force position interpolation, shift invariance for every shift, a from-scratch
 * complex-number route from the un-rotated inputs; "parity unpinned" against the paper, which prints no formula for it.
 * Not pinned by the paper: absolute output values (none are printed) and the RoPE
 * pairing convention (R5) -- "parity unpinned" for those two points only.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* Eq.(2): G = max(1, ceil(L / w_pretrained)), integer arithmetic only. */
int64_t jlo_group_size(int64_t L, int64_t w_pre) {
    if (L < 1 || w_pre < 1) return -1;
    int64_t G = (L + w_pre - 1) / w_pre;
    return G < 1 ? 1 : G;
}

/* Eq.(3): f(x) = floor(x / G), 0-based absolute positions (R2). */
int64_t jlo_remote_pos(int64_t x, int64_t G) { return x / G; }

/* Eq.(5): Delta(x) = f(x) - x. */
int64_t jlo_delta(int64_t x, int64_t G) { return x / G - x; }

/* theta_i = rope_theta^(-2i/d), i in [0, d/2)  (R5: "standard RoPE"). */
static double freq(double theta, int d, int i) { return pow(theta, -2.0 * (double)i / (double)d); }

/* RoPE(x, n): rotate every pair (x_i, x_{i+d/2}) by the angle n*theta_i (R5, half-split
 * pairing).  Used for Eq.(6) P:106 with n = Delta.  y may not alias x. */
static void rope_fr(const double* x, int d, const double* fr, int64_t n, double* y) {
    int h = d / 2;
    for (int i = 0; i < h; ++i) {
        double a = (double)n * fr[i];
        double c = cos(a), s = sin(a);
        y[i]     = x[i] * c - x[i + h] * s;
        y[i + h] = x[i] * s + x[i + h] * c;
    }
}
void jlo_rope(const double* x, int d, double theta, int64_t n, double* y) {
    double fr[4096];
    for (int i = 0; i < d / 2 && i < 4096; ++i) fr[i] = freq(theta, d, i);
    rope_fr(x, d, fr, n, y);
}

int jlo_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* One softmax over an explicit list of (score, value-row) terms: returns O and lse.
 * s[j] are the scaled scores, vrow[j] point at d floats.  Empty set: lse = -inf, O = 0. */
static void softmax_pv(const double* s, const float* const* vrow, int64_t cnt, int d,
                       double* O, double* lse) {
    for (int c = 0; c < d; ++c) O[c] = 0.0;
    if (cnt == 0) { *lse = -INFINITY; return; }
    double m = -INFINITY;
    for (int64_t j = 0; j < cnt; ++j) if (s[j] > m) m = s[j];
    double l = 0.0;
    for (int64_t j = 0; j < cnt; ++j) {
        double p = exp(s[j] - m);
        l += p;
        const float* v = vrow[j];
        for (int c = 0; c < d; ++c) O[c] += p * (double)v[c];
    }
    for (int c = 0; c < d; ++c) O[c] /= l;
    *lse = m + log(l);
}

static double dotd(const double* a, const double* b, int d) {
    double acc = 0.0;
    for (int c = 0; c < d; ++c) acc += a[c] * b[c];
    return acc;
}

/*
 * Direct definition (Eq.(1) P:70 with Eq.(2),(3),(5),(6)):
 *   s(q,k) = scale * <Qin[q], Kin[k]>                          if 0 <= q-k <= w0   (R1)
 *   s(q,k) = scale * <R(Delta q) Qin[q], R(Delta k) Kin[k]>    if q-k > w0
 *   out = softmax_k<=q(s) V,  lse = ln sum_k<=q exp(s),  scale = 1/sqrt(d)  (R7)
 * mode 0 = bifocal, mode 1 = plain causal control (first branch for every k <= q).
 * One G for all rows, from the full length L (R3).  GQA: kv head = h / (H_q/H_kv) (R9).
 * pos_shift shifts every absolute position (q and k) by a constant before Eq.(3)/(5); the
 * library contract is pos_shift = 0, the shift-invariance pin uses other values.
 * Ls (may be NULL): per-pair current sequence length L_j for decode runs; G_j = G(L_j).
 * Returns 0, or -1 on bad arguments.
 */
int jlo_attend_rows(const float* Qrows, const float* K, const float* V,
                    int64_t L, int H_q, int H_kv, int d,
                    int64_t w0, int64_t w_pre, double theta, int mode, int64_t pos_shift,
                    int64_t n, const int64_t* rows, const int32_t* heads, const int64_t* Ls,
                    double* out, double* lse) {
    if (L < 1 || H_q < 1 || H_kv < 1 || H_q % H_kv || d < 2 || (d & 1) || w0 < 0 || w_pre < 1 ||
        !(theta > 0.0) || n < 0) return -1;
    const int64_t G_all = jlo_group_size(L, w_pre);
    const int g = H_q / H_kv;
    const double scale = 1.0 / sqrt((double)d);
    double fr[4096];                       /* theta_i, i < d/2, computed once per call */
    if (d / 2 > 4096) return -1;
    for (int i = 0; i < d / 2; ++i) fr[i] = freq(theta, d, i);
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t j = 0; j < n; ++j) {
        const int64_t q = rows[j];
        const int h = heads[j];
        if (q < 0 || q >= L || h < 0 || h >= H_q) { bad = 1; continue; }
        /* decode runs: pair j may carry its own current length L_j <= L; G follows it (R4, R14) */
        int64_t G = G_all;
        if (Ls) { if (Ls[j] < 1 || Ls[j] > L || q >= Ls[j]) { bad = 1; continue; } G = jlo_group_size(Ls[j], w_pre); }
        const int kv = h / g;
        double* qloc = (double*)malloc(sizeof(double) * d * 3);
        double* qrem = qloc + d;
        double* kd = qrem + d;
        double* krem = (double*)malloc(sizeof(double) * d);
        double* s = (double*)malloc(sizeof(double) * (q + 1));
        const float** vrow = (const float**)malloc(sizeof(float*) * (q + 1));
        for (int c = 0; c < d; ++c) qloc[c] = (double)Qrows[j * d + c];
        rope_fr(qloc, d, fr, jlo_delta(q + pos_shift, G), qrem);       /* Eq.(6), query side */
        for (int64_t k = 0; k <= q; ++k) {
            const float* kp = K + ((size_t)k * H_kv + kv) * d;
            for (int c = 0; c < d; ++c) kd[c] = (double)kp[c];
            if (mode == 1 || q - k <= w0) {
                s[k] = scale * dotd(qloc, kd, d);                          /* Eq.(1), first case */
            } else {
                rope_fr(kd, d, fr, jlo_delta(k + pos_shift, G), krem); /* Eq.(6), key side */
                s[k] = scale * dotd(qrem, krem, d);                        /* Eq.(1), second case */
            }
            vrow[k] = V + ((size_t)k * H_kv + kv) * d;
        }
        softmax_pv(s, vrow, q + 1, d, out + j * d, lse + j);
        free(qloc); free(krem); free(s); free((void*)vrow);
    }
    return bad ? -1 : 0;
}

/*
 * Literal Section 3.3: three attention calls, each returning (O_X, l_X), then
 * Eq.(7).  A = sliding window (0 <= q-k <= w0), base q/k.  B = full causal, remote q/k.
 * C = sliding window, remote q/k.  M = max(l_A,l_B,l_C), W_X = exp(l_X - M),
 *   O = (W_A O_A + W_B O_B - W_C O_C) / (W_A + W_B - W_C),  lse = M + ln(W_A + W_B - W_C).
 * Rows with no remote key: B and C run over the same keys in the same order so that
 * W_B - W_C is exactly 0 (R13).  parts (optional, may be NULL): [n, 3] doubles = l_A,l_B,l_C.
 */
int jlo_three_call_rows(const float* Qrows, const float* K, const float* V,
                        int64_t L, int H_q, int H_kv, int d,
                        int64_t w0, int64_t w_pre, double theta,
                        int64_t n, const int64_t* rows, const int32_t* heads,
                        double* out, double* lse, double* parts) {
    if (L < 1 || H_q < 1 || H_kv < 1 || H_q % H_kv || d < 2 || (d & 1) || w0 < 0 || w_pre < 1 ||
        !(theta > 0.0) || n < 0) return -1;
    const int64_t G = jlo_group_size(L, w_pre);
    const int g = H_q / H_kv;
    const double scale = 1.0 / sqrt((double)d);
    double fr[4096];                       /* theta_i, i < d/2, computed once per call */
    if (d / 2 > 4096) return -1;
    for (int i = 0; i < d / 2; ++i) fr[i] = freq(theta, d, i);
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t j = 0; j < n; ++j) {
        const int64_t q = rows[j];
        const int h = heads[j];
        if (q < 0 || q >= L || h < 0 || h >= H_q) { bad = 1; continue; }
        const int kv = h / g;
        double* buf = (double*)malloc(sizeof(double) * d * 7);
        double *qloc = buf, *qrem = buf + d, *kd = buf + 2 * d, *krem = buf + 3 * d;
        double *OA = buf + 4 * d, *OB = buf + 5 * d, *OC = buf + 6 * d;
        double* sA = (double*)malloc(sizeof(double) * (q + 1) * 3);
        double *sB = sA + (q + 1), *sC = sB + (q + 1);
        const float** vA = (const float**)malloc(sizeof(float*) * (q + 1) * 3);
        const float **vB = vA + (q + 1), **vC = vB + (q + 1);
        int64_t nA = 0, nB = 0, nC = 0;
        for (int c = 0; c < d; ++c) qloc[c] = (double)Qrows[j * d + c];
        rope_fr(qloc, d, fr, jlo_delta(q, G), qrem);
        /* keys visited from the newest to the oldest so that, when every key is inside the
         * window, calls B and C sum the same terms in the same order (R13). */
        for (int64_t k = q; k >= 0; --k) {
            const float* kp = K + ((size_t)k * H_kv + kv) * d;
            const float* vp = V + ((size_t)k * H_kv + kv) * d;
            for (int c = 0; c < d; ++c) kd[c] = (double)kp[c];
            rope_fr(kd, d, fr, jlo_delta(k, G), krem);
            const double srem = scale * dotd(qrem, krem, d);
            sB[nB] = srem; vB[nB++] = vp;                                  /* call B */
            if (q - k <= w0) {
                sA[nA] = scale * dotd(qloc, kd, d); vA[nA++] = vp;         /* call A */
                sC[nC] = srem; vC[nC++] = vp;                              /* call C */
            }
        }
        double lA, lB, lC;
        softmax_pv(sA, vA, nA, d, OA, &lA);
        softmax_pv(sB, vB, nB, d, OB, &lB);
        softmax_pv(sC, vC, nC, d, OC, &lC);
        double M = lA; if (lB > M) M = lB; if (lC > M) M = lC;
        const double WA = exp(lA - M), WB = exp(lB - M), WC = exp(lC - M);
        const double den = WA + WB - WC;
        for (int c = 0; c < d; ++c) out[j * d + c] = (WA * OA[c] + WB * OB[c] - WC * OC[c]) / den;  /* Eq.(7) */
        lse[j] = M + log(den);
        if (parts) { parts[j * 3] = lA; parts[j * 3 + 1] = lB; parts[j * 3 + 2] = lC; }
        free(buf); free(sA); free((void*)vA);
    }
    return bad ? -1 : 0;
}

/* Scores only (no softmax): s[k] for k = 0..q of one (row, head); used by the closed-form
 * and aliasing pins.  Same rule as jlo_attend_rows. */
int jlo_scores_row(const float* Qrow, const float* K, int64_t L, int H_kv, int kv, int d,
                   int64_t w0, int64_t w_pre, double theta, int mode, int64_t q, double* s) {
    if (q < 0 || q >= L || (d & 1)) return -1;
    const int64_t G = jlo_group_size(L, w_pre);
    const double scale = 1.0 / sqrt((double)d);
    double fr[4096];
    if (d / 2 > 4096) return -1;
    for (int i = 0; i < d / 2; ++i) fr[i] = freq(theta, d, i);
    double* buf = (double*)malloc(sizeof(double) * d * 4);
    double *qloc = buf, *qrem = buf + d, *kd = buf + 2 * d, *krem = buf + 3 * d;
    for (int c = 0; c < d; ++c) qloc[c] = (double)Qrow[c];
    rope_fr(qloc, d, fr, jlo_delta(q, G), qrem);
    for (int64_t k = 0; k <= q; ++k) {
        const float* kp = K + ((size_t)k * H_kv + kv) * d;
        for (int c = 0; c < d; ++c) kd[c] = (double)kp[c];
        if (mode == 1 || q - k <= w0) s[k] = scale * dotd(qloc, kd, d);
        else { rope_fr(kd, d, fr, jlo_delta(k, G), krem); s[k] = scale * dotd(qrem, krem, d); }
    }
    free(buf);
    return 0;
}

/*
 * the "YaRN-style frequency interpolation" remote map "within the same bifocal
 * construction".  The paper prints no formula; reading R17 fixes it as NTK-by-parts (YaRN) with scale s = G:
 *   rotations of pair i inside the pretrained window   r_i = w_pre * theta_i / (2 pi)
 *   ramp                                               gamma_i = clamp((r_i - alpha) / (beta - alpha), 0, 1)
 *   remote frequency                                   theta'_i = theta_i * ((1 - gamma_i) / G + gamma_i)
 * and the remote branch of Eq.(1) scores RoPE at the TRUE positions with theta' instead of theta:
 *   s(q,k) = scale * <RoPE_theta'(x_q, q), RoPE_theta'(x_k, k)>                      if q-k > w0.
 * On the stored operands (RoPE_theta at true positions, Eq.(4)) that is the correction rotation of pair i by the
 * angle -x * phi_i, phi_i = theta_i - theta'_i = theta_i (1 - gamma_i)(1 - 1/G), x = the absolute position -- the analogue
 * of Eq.(6) with a per-frequency, non-integer Delta_i(x) = -x (1 - gamma_i)(1 - 1/G).  No extra temperature (R10).
 * G = 1 gives phi = 0 (the control); gamma = 1 everywhere gives the control; gamma = 0 everywhere is position
 * interpolation x -> x / G, which agrees with aliasing (Eq.(3)) at multiples of G.
 * Same layouts and conventions as jlo_attend_rows (mode is always bifocal).
 */
int jlo_attend_rows_freq(const float* Qrows, const float* K, const float* V,
                         int64_t L, int H_q, int H_kv, int d,
                         int64_t w0, int64_t w_pre, double theta, double alpha, double beta, int64_t pos_shift,
                         int64_t n, const int64_t* rows, const int32_t* heads,
                         double* out, double* lse) {
    if (L < 1 || H_q < 1 || H_kv < 1 || H_q % H_kv || d < 2 || (d & 1) || w0 < 0 || w_pre < 1 ||
        !(theta > 0.0) || n < 0 || !(beta > alpha) || d / 2 > 4096) return -1;
    const int64_t G = jlo_group_size(L, w_pre);
    const int g = H_q / H_kv, hd = d / 2;
    const double scale = 1.0 / sqrt((double)d);
    const double two_pi = 6.283185307179586476925286766559;
    double phi[4096];
    for (int i = 0; i < hd; ++i) {
        const double th = freq(theta, d, i);
        const double r = (double)w_pre * th / two_pi;
        double gam = (r - alpha) / (beta - alpha);
        gam = gam < 0.0 ? 0.0 : (gam > 1.0 ? 1.0 : gam);
        phi[i] = th * (1.0 - gam) * (1.0 - 1.0 / (double)G);
    }
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t j = 0; j < n; ++j) {
        const int64_t q = rows[j];
        const int h = heads[j];
        if (q < 0 || q >= L || h < 0 || h >= H_q) { bad = 1; continue; }
        const int kv = h / g;
        double* buf = (double*)malloc(sizeof(double) * d * 4);
        double *qloc = buf, *qrem = buf + d, *kd = buf + 2 * d, *krem = buf + 3 * d;
        double* s = (double*)malloc(sizeof(double) * (q + 1));
        const float** vrow = (const float**)malloc(sizeof(float*) * (q + 1));
        for (int c = 0; c < d; ++c) qloc[c] = (double)Qrows[j * d + c];
        for (int i = 0; i < hd; ++i) {                                  /* correction of the query: angle -(q) phi_i */
            const double a = -(double)(q + pos_shift) * phi[i], c = cos(a), sn = sin(a);
            qrem[i] = qloc[i] * c - qloc[i + hd] * sn;
            qrem[i + hd] = qloc[i] * sn + qloc[i + hd] * c;
        }
        for (int64_t k = 0; k <= q; ++k) {
            const float* kp = K + ((size_t)k * H_kv + kv) * d;
            for (int c = 0; c < d; ++c) kd[c] = (double)kp[c];
            if (q - k <= w0) {
                s[k] = scale * dotd(qloc, kd, d);                        /* Eq.(1), first case, unchanged */
            } else {
                for (int i = 0; i < hd; ++i) {                          /* correction of the key: angle -(k) phi_i */
                    const double a = -(double)(k + pos_shift) * phi[i], c = cos(a), sn = sin(a);
                    krem[i] = kd[i] * c - kd[i + hd] * sn;
                    krem[i + hd] = kd[i] * sn + kd[i + hd] * c;
                }
                s[k] = scale * dotd(qrem, krem, d);
            }
            vrow[k] = V + ((size_t)k * H_kv + kv) * d;
        }
        softmax_pv(s, vrow, q + 1, d, out + j * d, lse + j);
        free(buf); free(s); free((void*)vrow);
    }
    return bad ? -1 : 0;
}
