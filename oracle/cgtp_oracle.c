/*
 * cgtp_oracle.c -- FP64 CPU ORACLE for the contracted Clebsch-Gordan tensor product.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and the cpu_baseline /
 * --impl reference legs of bench.py may build, load or call this file.  The product path
 * (paper_2605_15073_b200/) never does and shares no code, header, table or constant with it.
 *
 * What it computes (citations are PAPER.md lines = /root/reference/PAPER.md):
 *   - on-site bilinear contraction Eq.(1) at fixed CP rank Eq.(3) (:39), for
 *     natural-parity inputs: "even" rank channels couple through the Gaunt coefficient Eq.(4)-(5)
 *     (:49-:55), "odd" rank channels through the surface-curl coefficient Q = kappa^-1 * G,
 *     Eq.(13)-(14) (:115-:119) with kappa^-1 from Eq.(A10) (:580).
 *   - message-passing coupling Eq.(2) (:33): edge factor R~[e,c] * Y_{l1 m1}(r_hat_e) (factor 1)
 *     times the sender's projected node feature (factor 2), summed over the in-edges of every
 *     receiver (Eq.(52) :415, Eq.(57) :443).
 * The method reaches these sums exactly (the grid quadrature is exact), so the oracle is the plain
 * definition written out as a direct sparse sum over closed-form coefficients.  Nothing in this
 * file touches a quadrature grid.
 *
 * Readings of the paper used here:
 *   R1  spherical harmonics are orthonormal on S^2.
 *   R2  real basis of Eq.(C1) (:663) without Condon-Shortley phase, order m=-l..l, flat index
 *       l*l+l+m; (Y_{1,-1},Y_{1,0},Y_{1,1}) = sqrt(3/4pi) (y,z,x).
 *   R4  with given weights the pipeline realises the Gaunt-weighted (even) / Q-weighted (odd)
 *       coupling (the prefactors f, kappa are absorbed in the learnable weights, :157, :374-:381).
 *   R5  l-shared weights W_a,W_b[C,N], W_out[N,C].   R6  parity_mask[c]: 0 even, 1 odd; two output
 *       sectors.   R10 bracket {1,2} = d_phi A1 d_x A2 - d_x A1 d_phi A2, on-site A is factor 1,
 *       message passing: edge is factor 1.   R11 edge_vec = r_j - r_i, edge_index row 0 sender,
 *       row 1 receiver, receiver-sorted.   R12 l1-shared radial factor edge_radial[E,C].
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): Wigner 3j and Gaunt against sympy's exact values,
 * Eq.(6) closed form, the printed kappa^-1 values (:600, :655) and worked example (A11)-(A13),
 * real-basis tables against brute-force quadrature, (1,1,1) block = sqrt(3/4pi)*epsilon,
 * real SH against scipy, whole-pipeline results against fine-grid quadrature, Wigner-D
 * equivariance, inversion parity, self-coupled vanishing, Parseval; the parity-slot functions
 * (oracle_*_parity) against the paper's dispatch check B7 (:647), the reduction to the natural-parity
 * functions, Eq.(44)-(45)/(56) slot rules, inversion and rotation; the l-dependent-weight functions
 * (oracle_*_lw) against the l-shared functions (equal weights, degree selection, per-degree numpy
 * projections around them) and rotation; the nu-body function (oracle_onsite_nbody) against fine-grid
 * quadrature of the pointwise product, the closed form Y_10^3 = (3/4pi)^(3/2) (3/5 z + 2/5 P_3(z)), the
 * reduction to oracle_onsite at nu = 2, factor permutation and rotation (tests/test_oracle_nbody.py); the
 * two-field function (oracle_message_field, Eq.(28)) against oracle_message for edge fields of the form R.Y,
 * fine-grid quadrature of the pooled pointwise product, one-edge receivers = oracle_onsite, edge order inside a
 * segment and rotation, and its l-dependent-weight form (oracle_message_field_lw) against it (equal weights, degree
 * selection, per-degree numpy projections around it) (tests/test_oracle_field.py).
 * oracle_message_field_parity (Eq.(28) with the parity labels of both fields, Sec. VII C f :471) is pinned
 * (tests/test_oracle_field_parity.py) to oracle_message_field per run (one slot pair populated), to oracle_onsite_parity on
 * one-edge receivers, to B7-style exact vanishing in the wrong sector (:647), to inversion with the slots' labels and to
 * Wigner-D rotation.
 * No function here is "parity unpinned".
 *
 * Plain C99 + OpenMP, double precision (long double inside the Racah sum).
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846264338327950288
#endif

/* ------------------------------------------------------------------------------------------ */
/* Angular-momentum algebra                                                                   */
/* ------------------------------------------------------------------------------------------ */

static long double lfact(int n) { return lgammal((long double)n + 1.0L); }

static int triangle_ok(int a, int b, int c) { return c >= abs(a - b) && c <= a + b; }

/* Wigner 3j symbol (j1 j2 j3; m1 m2 m3), integer arguments, Racah's single-sum formula
 * (the "standard 3-j/CG relation" the paper invokes at :578; ref. [41] of the paper). */
double oracle_wigner3j(int j1, int j2, int j3, int m1, int m2, int m3)
{
    if (j1 < 0 || j2 < 0 || j3 < 0) return 0.0;
    if (m1 + m2 + m3 != 0) return 0.0;
    if (abs(m1) > j1 || abs(m2) > j2 || abs(m3) > j3) return 0.0;
    if (!triangle_ok(j1, j2, j3)) return 0.0;
    long double logpref = 0.5L * (lfact(j1 + j2 - j3) + lfact(j1 - j2 + j3) + lfact(-j1 + j2 + j3)
                                  - lfact(j1 + j2 + j3 + 1)
                                  + lfact(j1 + m1) + lfact(j1 - m1) + lfact(j2 + m2) + lfact(j2 - m2)
                                  + lfact(j3 + m3) + lfact(j3 - m3));
    int tmin = 0;
    if (j2 - j3 - m1 > tmin) tmin = j2 - j3 - m1;
    if (j1 - j3 + m2 > tmin) tmin = j1 - j3 + m2;
    int tmax = j1 + j2 - j3;
    if (j1 - m1 < tmax) tmax = j1 - m1;
    if (j2 + m2 < tmax) tmax = j2 + m2;
    long double sum = 0.0L;
    for (int t = tmin; t <= tmax; ++t) {
        long double logden = lfact(t) + lfact(j3 - j2 + t + m1) + lfact(j3 - j1 + t - m2)
                             + lfact(j1 + j2 - j3 - t) + lfact(j1 - t - m1) + lfact(j2 - t + m2);
        long double term = expl(logpref - logden);
        sum += (t & 1) ? -term : term;
    }
    int ph = j1 - j2 - m3;
    if (ph & 1) sum = -sum;
    return (double)sum;
}

/* Clebsch-Gordan coefficient G^{l m}_{l1 m1 l2 m2} = <l1 m1 l2 m2 | l m> (Condon-Shortley). */
double oracle_cg(int l1, int m1, int l2, int m2, int l, int m)
{
    if (m1 + m2 != m) return 0.0;
    double w = oracle_wigner3j(l1, l2, l, m1, m2, -m);
    int ph = l1 - l2 + m;
    double s = (ph & 1) ? -1.0 : 1.0;
    return s * sqrt(2.0 * l + 1.0) * w;
}

/* Eq.(6)-(7) (PAPER.md:59-:63): closed form of G^{l0}_{l1 0 l2 0}; Eq.(8) (:70): zero for odd sum. */
double oracle_cg000_closed(int l1, int l2, int l)
{
    if (!triangle_ok(l1, l2, l)) return 0.0;
    int s = l1 + l2 + l;
    if (s & 1) return 0.0;
    int g = s / 2;
    long double logdelta = lfact(l1 + l2 - l) + lfact(l1 - l2 + l) + lfact(-l1 + l2 + l) - lfact(s + 1);
    long double logv = 0.5L * logdelta + lfact(g) - lfact(g - l1) - lfact(g - l2) - lfact(g - l);
    double v = sqrt(2.0 * l + 1.0) * (double)expl(logv);
    int ph = l1 - l2 + g;
    return (ph & 1) ? -v : v;
}

/* Eq.(4)-(5) (PAPER.md:49-:55): complex Gaunt coefficient  int Y_{l1m1} Y_{l2m2} Y*_{lm} dOmega. */
double oracle_gaunt_complex(int l1, int m1, int l2, int m2, int l, int m)
{
    if (m1 + m2 != m) return 0.0;
    double g0 = oracle_cg000_closed(l1, l2, l);
    if (g0 == 0.0) return 0.0;
    double pref = sqrt((2.0 * l1 + 1.0) * (2.0 * l2 + 1.0) / (4.0 * M_PI * (2.0 * l + 1.0)));
    return pref * g0 * oracle_cg(l1, m1, l2, m2, l, m);
}

/* Eq.(A10): kappa^-1(l1,l2,l) is purely imaginary in the complex basis; this returns
 * its imaginary part, i.e. kappa^-1 = i * oracle_kappa_inv_imag.  Support (:583-:585): l1,l2>=1,
 * triangle, l1+l2+l odd; zero elsewhere (Eq.(A7) :560). */
double oracle_kappa_inv_imag(int l1, int l2, int l)
{
    if (l1 < 1 || l2 < 1 || !triangle_ok(l1, l2, l)) return 0.0;
    if (((l1 + l2 + l) & 1) == 0) return 0.0;
    double pref = sqrt((2.0 * l1 + 1.0) * (2.0 * l2 + 1.0) * l1 * (l1 + 1.0) * l2 * (l2 + 1.0) / (4.0 * M_PI));
    double w = oracle_wigner3j(l1, l2, l, -1, 1, 0);
    int ph = l1 - l2;
    double s = (ph & 1) ? -1.0 : 1.0;
    /* kappa^-1 = -i * (-1)^{l1-l2} * pref * 3j  ->  imaginary part = -(-1)^{l1-l2} pref 3j */
    return -s * pref * w;
}

/* Eq.(13)-(14) (PAPER.md:115-:119): complex surface-curl coefficient Q = kappa^-1 * G (purely
 * imaginary); returns its imaginary part. */
double oracle_q_complex_imag(int l1, int m1, int l2, int m2, int l, int m)
{
    if (m1 + m2 != m) return 0.0;
    double k = oracle_kappa_inv_imag(l1, l2, l);
    if (k == 0.0) return 0.0;
    return k * oracle_cg(l1, m1, l2, m2, l, m);
}

/* ------------------------------------------------------------------------------------------ */
/* Complex -> real basis (reading R2; Eq.(C1), complex CS basis as in App. B :611) */
/*   m>0 : Y^r_{l,m}  = ((-1)^m Y^c_{l,m} + Y^c_{l,-m}) / sqrt2                                 */
/*   m=0 : Y^r_{l,0}  = Y^c_{l,0}                                                               */
/*   m<0 : Y^r_{l,m}  = ((-1)^a Y^c_{l,a} - Y^c_{l,-a}) / (i sqrt2),  a=|m|                      */
/* U(m, mu) is the coefficient of Y^c_{l,mu} in Y^r_{l,m}; only mu = +-|m| are non-zero.         */
/* ------------------------------------------------------------------------------------------ */
static double complex real_from_complex_U(int m, int mu)
{
    const double r = 0.70710678118654752440;
    if (m == 0) return (mu == 0) ? 1.0 : 0.0;
    int a = abs(m);
    if (abs(mu) != a) return 0.0;
    double sa = (a & 1) ? -1.0 : 1.0;
    if (m > 0) return (mu > 0) ? sa * r : r;
    /* m<0: 1/(i sqrt2) = -i/sqrt2 */
    return (mu > 0) ? (-I * sa * r) : (I * r);
}

typedef struct {
    int lmax, lmax_out, odd;
    int64_t nnz;
    int32_t *i1, *i2, *io;
    double *val;
    double max_imag; /* largest discarded imaginary part (must be round-off) */
} coupling_t;

#define MAX_CACHED 512
static coupling_t g_cache[MAX_CACHED];
static int g_ncache = 0;

/* Real-basis coupling tensor, sparse COO:
 *   odd=0:  Gr(a,b;c) = int Y_a Y_b Y_c dOmega                  (real Gaunt; Eq.(4)-(5) in the real basis)
 *   odd=1:  Qr(a,b;c) = int r.[grad Y_a x grad Y_b] Y_c dOmega  (Eq.(13) in the real basis)
 * via T^r_{abc} = sum U1(a,mu1) U2(b,mu2) conj(U3(c,mu)) T^c(mu1,mu2;mu). */
static const coupling_t *get_coupling(int lmax, int lmax_out, int odd)
{
    const coupling_t *found = NULL;
#pragma omp critical(cgtp_oracle_cache)
    {
        for (int i = 0; i < g_ncache; ++i)
            if (g_cache[i].lmax == lmax && g_cache[i].lmax_out == lmax_out && g_cache[i].odd == odd)
                found = &g_cache[i];
        if (!found && g_ncache < MAX_CACHED) {
            coupling_t t;
            memset(&t, 0, sizeof t);
            t.lmax = lmax; t.lmax_out = lmax_out; t.odd = odd;
            int64_t cap = 1024;
            t.i1 = malloc(cap * sizeof(int32_t)); t.i2 = malloc(cap * sizeof(int32_t));
            t.io = malloc(cap * sizeof(int32_t)); t.val = malloc(cap * sizeof(double));
            int W = 2 * lmax + 1;
            double *tc = malloc((size_t)W * W * sizeof(double)); /* complex-basis table at fixed (l1,l2,l) */
            for (int l1 = 0; l1 <= lmax; ++l1)
            for (int l2 = 0; l2 <= lmax; ++l2)
            for (int l = abs(l1 - l2); l <= l1 + l2 && l <= lmax_out; ++l) {
                int par = (l1 + l2 + l) & 1;
                if (par != odd) continue;
                if (odd && (l1 < 1 || l2 < 1)) continue;
                /* complex table: real number g (even) or imaginary part q (odd: value = i*q) */
                for (int m1 = -l1; m1 <= l1; ++m1)
                for (int m2 = -l2; m2 <= l2; ++m2) {
                    int m = m1 + m2;
                    double v = 0.0;
                    if (abs(m) <= l)
                        v = odd ? oracle_q_complex_imag(l1, m1, l2, m2, l, m)
                                : oracle_gaunt_complex(l1, m1, l2, m2, l, m);
                    tc[(m1 + l1) * W + (m2 + l2)] = v;
                }
                for (int a = -l1; a <= l1; ++a)
                for (int b = -l2; b <= l2; ++b)
                for (int c = -l; c <= l; ++c) {
                    double complex acc = 0.0;
                    for (int s1 = 0; s1 < 2; ++s1) {
                        int mu1 = s1 ? -abs(a) : abs(a);
                        if (a == 0 && s1) continue;
                        double complex u1 = real_from_complex_U(a, mu1);
                        for (int s2 = 0; s2 < 2; ++s2) {
                            int mu2 = s2 ? -abs(b) : abs(b);
                            if (b == 0 && s2) continue;
                            int mu = mu1 + mu2;
                            if (abs(mu) != abs(c)) continue;
                            double complex u2 = real_from_complex_U(b, mu2);
                            double complex u3 = real_from_complex_U(c, mu);
                            double v = tc[(mu1 + l1) * W + (mu2 + l2)];
                            double complex tcv = odd ? (I * v) : v;
                            acc += u1 * u2 * conj(u3) * tcv;
                        }
                    }
                    if (fabs(cimag(acc)) > t.max_imag) t.max_imag = fabs(cimag(acc));
                    double r = creal(acc);
                    if (fabs(r) > 1e-12) {
                        if (t.nnz == cap) {
                            cap *= 2;
                            t.i1 = realloc(t.i1, cap * sizeof(int32_t)); t.i2 = realloc(t.i2, cap * sizeof(int32_t));
                            t.io = realloc(t.io, cap * sizeof(int32_t)); t.val = realloc(t.val, cap * sizeof(double));
                        }
                        t.i1[t.nnz] = l1 * l1 + l1 + a;
                        t.i2[t.nnz] = l2 * l2 + l2 + b;
                        t.io[t.nnz] = l * l + l + c;
                        t.val[t.nnz] = r;
                        t.nnz++;
                    }
                }
            }
            free(tc);
            g_cache[g_ncache] = t;
            found = &g_cache[g_ncache];
            g_ncache++;
        }
    }
    return found;
}

/* Exported view of the real-basis coupling tensor.  Call with NULL arrays to get nnz. */
int64_t oracle_real_coupling(int lmax, int lmax_out, int odd, int32_t *i1, int32_t *i2, int32_t *io,
                             double *val, double *max_imag)
{
    const coupling_t *t = get_coupling(lmax, lmax_out, odd);
    if (!t) return -1;
    if (max_imag) *max_imag = t->max_imag;
    if (i1 && i2 && io && val) {
        memcpy(i1, t->i1, t->nnz * sizeof(int32_t));
        memcpy(i2, t->i2, t->nnz * sizeof(int32_t));
        memcpy(io, t->io, t->nnz * sizeof(int32_t));
        memcpy(val, t->val, t->nnz * sizeof(double));
    }
    return t->nnz;
}

/* ------------------------------------------------------------------------------------------ */
/* Real spherical harmonics of a direction (reading R1/R2), needed for the edge feature         */
/* R(r) Y_{l1 m1}(r_hat) of Eq.(2) (PAPER.md:33-:35).                                           */
/*   Y_{lm} = sqrt2 Pt_l^{|m|}(cos th) cos(m ph)  (m>0),  Pt_l^0  (m=0),  sqrt2 Pt sin(|m| ph) (m<0) */
/*   Pt_l^m = sqrt((2l+1)/(4pi) (l-m)!/(l+m)!) P_l^m,  P_l^m WITHOUT the Condon-Shortley phase.  */
/* ------------------------------------------------------------------------------------------ */
void oracle_real_sh(int lmax, double x, double y, double z, double *Y /* [(lmax+1)^2] */)
{
    double r = sqrt(x * x + y * y + z * z);
    double ct = z / r;
    double st = sqrt(x * x + y * y) / r;
    double ph = atan2(y, x);
    int L = lmax + 1;
    double *P = calloc((size_t)L * L, sizeof(double)); /* P[l*L+m] = Pt_l^m */
    /* sectoral seeds Pt_m^m, then the standard three-term upward recurrence in l */
    P[0] = sqrt(1.0 / (4.0 * M_PI));
    for (int m = 1; m <= lmax; ++m)
        P[m * L + m] = sqrt((2.0 * m + 1.0) / (2.0 * m)) * st * P[(m - 1) * L + (m - 1)];
    for (int m = 0; m <= lmax; ++m) {
        if (m + 1 <= lmax) P[(m + 1) * L + m] = sqrt(2.0 * m + 3.0) * ct * P[m * L + m];
        for (int l = m + 2; l <= lmax; ++l) {
            double a = sqrt((4.0 * l * l - 1.0) / ((double)l * l - (double)m * m));
            double b = sqrt((((double)l - 1.0) * (l - 1.0) - (double)m * m) / (4.0 * (l - 1.0) * (l - 1.0) - 1.0));
            P[l * L + m] = a * (ct * P[(l - 1) * L + m] - b * P[(l - 2) * L + m]);
        }
    }
    const double s2 = sqrt(2.0);
    for (int l = 0; l <= lmax; ++l) {
        Y[l * l + l] = P[l * L];
        for (int m = 1; m <= l; ++m) {
            Y[l * l + l + m] = s2 * P[l * L + m] * cos(m * ph);
            Y[l * l + l - m] = s2 * P[l * L + m] * sin(m * ph);
        }
    }
    free(P);
}

/* ------------------------------------------------------------------------------------------ */
/* Segmentation (integer work): CSR offsets of a receiver-sorted edge list.                     */
/* row_ptr[i] = first edge whose receiver is >= i;  row_ptr[nodes] = E.                         */
/* Returns 0 if valid, 4 if not sorted / out of range (same code as the library's error 4).     */
/* ------------------------------------------------------------------------------------------ */
int oracle_segments(const int64_t *edge_index /* [2,E] */, int64_t E, int64_t nodes, int64_t *row_ptr)
{
    const int64_t *snd = edge_index, *rcv = edge_index + E;
    for (int64_t e = 0; e < E; ++e) {
        if (rcv[e] < 0 || rcv[e] >= nodes || snd[e] < 0 || snd[e] >= nodes) return 4;
        if (e > 0 && rcv[e] < rcv[e - 1]) return 4;
    }
    int64_t e = 0;
    for (int64_t i = 0; i <= nodes; ++i) {
        while (e < E && rcv[e] < i) ++e;
        row_ptr[i] = e;
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* On-site contraction, Eq.(1) with the CP factorisation Eq.(3).                                */
/*   Ha[c,:] = W_a[c,:] . A[b]      Hb[c,:] = W_b[c,:] . B[b]                  (Eq.(35) :322)   */
/*   T[c,lm] = sum coef(i1,i2;lm) Ha[c,i1] Hb[c,i2]   coef = Gr (mask 0) or Qr (mask 1)         */
/*   out[b,s,n,lm] = sum_{c: mask[c]=s} W_out[n,c] T[c,lm]                     (Eq.(41) :346)   */
/* Layouts: A,B [batch,N,(lmax+1)^2]; W_a,W_b [C,N]; W_out [N,C]; out [batch,2,N,(lmax_out+1)^2] */
/* ------------------------------------------------------------------------------------------ */
int oracle_onsite(const double *A, const double *B, const double *W_a, const double *W_b,
                  const double *W_out, int lmax, int lmax_out, int N, int C, const uint8_t *parity_mask,
                  double *out, int64_t batch)
{
    int L2 = (lmax + 1) * (lmax + 1), Lo2 = (lmax_out + 1) * (lmax_out + 1);
    const coupling_t *tab[2];
    tab[0] = get_coupling(lmax, lmax_out, 0);
    tab[1] = get_coupling(lmax, lmax_out, 1);
    if (!tab[0] || !tab[1]) return 2;
#pragma omp parallel
    {
        double *Ha = malloc((size_t)C * L2 * sizeof(double));
        double *Hb = malloc((size_t)C * L2 * sizeof(double));
        double *T = malloc((size_t)C * Lo2 * sizeof(double));
#pragma omp for schedule(dynamic, 1)
        for (int64_t b = 0; b < batch; ++b) {
            const double *Ab = A + b * (int64_t)N * L2, *Bb = B + b * (int64_t)N * L2;
            for (int c = 0; c < C; ++c)
                for (int i = 0; i < L2; ++i) {
                    double sa = 0.0, sb = 0.0;
                    for (int n = 0; n < N; ++n) {
                        sa += W_a[c * N + n] * Ab[n * L2 + i];
                        sb += W_b[c * N + n] * Bb[n * L2 + i];
                    }
                    Ha[c * L2 + i] = sa;
                    Hb[c * L2 + i] = sb;
                }
            for (int c = 0; c < C; ++c) {
                const coupling_t *t = tab[parity_mask[c] ? 1 : 0];
                double *Tc = T + (size_t)c * Lo2;
                const double *ha = Ha + (size_t)c * L2, *hb = Hb + (size_t)c * L2;
                for (int i = 0; i < Lo2; ++i) Tc[i] = 0.0;
                for (int64_t k = 0; k < t->nnz; ++k)
                    Tc[t->io[k]] += t->val[k] * ha[t->i1[k]] * hb[t->i2[k]];
            }
            double *ob = out + b * 2 * (int64_t)N * Lo2;
            for (int s = 0; s < 2; ++s)
                for (int n = 0; n < N; ++n)
                    for (int i = 0; i < Lo2; ++i) {
                        double acc = 0.0;
                        for (int c = 0; c < C; ++c)
                            if ((parity_mask[c] ? 1 : 0) == s) acc += W_out[n * C + c] * T[(size_t)c * Lo2 + i];
                        ob[((size_t)s * N + n) * Lo2 + i] = acc;
                    }
        }
        free(Ha); free(Hb); free(T);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* Message passing, Eq.(2) with the CP factorisation Eq.(42)-(43) and the l1-shared radial      */
/* factor (reading R12).  For receiver i with in-edges e (sender j = send(e)):                  */
/*   a[e,c,l1m1] = edge_radial[e,c] * Y_{l1m1}(edge_vec[e]/|edge_vec[e]|)   (factor 1, Eq.(46),(48)) */
/*   H[j,c,:]    = W_node[c,:] . node_feats[j]                              (factor 2, Eq.(47))  */
/*   T[i,c,lm]   = sum_e sum coef(i1,i2;lm) a[e,c,i1] H[j,c,i2]             (Eq.(52) / Eq.(57))  */
/*   out[i,s,n,lm] = sum_{c: mask[c]=s} W_out[n,c] T[i,c,lm]                (Eq.(55),(58),(59))  */
/* recv_list/n_recv select the receivers that are evaluated (NULL = all nodes); out has one      */
/* block [2,N,(lmax_out+1)^2] per evaluated receiver, in list order.                             */
/* ------------------------------------------------------------------------------------------ */
int oracle_message(const double *node_feats /* [nodes,N,L2] */, const int64_t *edge_index /* [2,E] */,
                   const double *edge_vec /* [E,3] */, const double *edge_radial /* [E,C] */,
                   const double *W_node /* [C,N] */, const double *W_out /* [N,C] */,
                   int lmax, int lmax_out, int N, int C, const uint8_t *parity_mask,
                   double *out, int64_t nodes, int64_t E, const int64_t *recv_list, int64_t n_recv)
{
    int L2 = (lmax + 1) * (lmax + 1), Lo2 = (lmax_out + 1) * (lmax_out + 1);
    const coupling_t *tab[2];
    tab[0] = get_coupling(lmax, lmax_out, 0);
    tab[1] = get_coupling(lmax, lmax_out, 1);
    if (!tab[0] || !tab[1]) return 2;
    int64_t *row_ptr = malloc((size_t)(nodes + 1) * sizeof(int64_t));
    int rc = oracle_segments(edge_index, E, nodes, row_ptr);
    if (rc) { free(row_ptr); return rc; }
    const int64_t *snd = edge_index;
    int64_t nr = recv_list ? n_recv : nodes;
    /* Eq.(47): project only the senders that the evaluated receivers need (once per node). */
    int64_t *slot = malloc((size_t)nodes * sizeof(int64_t));
    for (int64_t j = 0; j < nodes; ++j) slot[j] = -1;
    int64_t n_need = 0;
    for (int64_t r = 0; r < nr; ++r) {
        int64_t i = recv_list ? recv_list[r] : r;
        for (int64_t e = row_ptr[i]; e < row_ptr[i + 1]; ++e)
            if (slot[snd[e]] < 0) slot[snd[e]] = n_need++;
    }
    double *H = malloc((size_t)(n_need > 0 ? n_need : 1) * C * L2 * sizeof(double));
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t j = 0; j < nodes; ++j) {
        if (slot[j] < 0) continue;
        const double *xj = node_feats + j * (int64_t)N * L2;
        double *hj = H + slot[j] * (int64_t)C * L2;
        for (int c = 0; c < C; ++c)
            for (int q = 0; q < L2; ++q) {
                double s = 0.0;
                for (int n = 0; n < N; ++n) s += W_node[c * N + n] * xj[n * L2 + q];
                hj[c * L2 + q] = s;
            }
    }
#pragma omp parallel
    {
        double *Y = malloc((size_t)L2 * sizeof(double));
        double *a = malloc((size_t)L2 * sizeof(double));
        double *T = malloc((size_t)C * Lo2 * sizeof(double));
#pragma omp for schedule(dynamic, 1)
        for (int64_t r = 0; r < nr; ++r) {
            int64_t i = recv_list ? recv_list[r] : r;
            for (size_t k = 0; k < (size_t)C * Lo2; ++k) T[k] = 0.0;
            for (int64_t e = row_ptr[i]; e < row_ptr[i + 1]; ++e) {
                const double *hj = H + slot[snd[e]] * (int64_t)C * L2;
                oracle_real_sh(lmax, edge_vec[3 * e], edge_vec[3 * e + 1], edge_vec[3 * e + 2], Y);
                for (int c = 0; c < C; ++c) {
                    double rad = edge_radial[e * (int64_t)C + c];
                    for (int q = 0; q < L2; ++q) a[q] = rad * Y[q];
                    const double *h = hj + (size_t)c * L2;
                    const coupling_t *t = tab[parity_mask[c] ? 1 : 0];
                    double *Tc = T + (size_t)c * Lo2;
                    for (int64_t k = 0; k < t->nnz; ++k)
                        Tc[t->io[k]] += t->val[k] * a[t->i1[k]] * h[t->i2[k]];
                }
            }
            double *ob = out + r * 2 * (int64_t)N * Lo2;
            for (int s = 0; s < 2; ++s)
                for (int n = 0; n < N; ++n)
                    for (int q = 0; q < Lo2; ++q) {
                        double acc = 0.0;
                        for (int c = 0; c < C; ++c)
                            if ((parity_mask[c] ? 1 : 0) == s) acc += W_out[n * C + c] * T[(size_t)c * Lo2 + q];
                        ob[((size_t)s * N + n) * Lo2 + q] = acc;
                    }
        }
        free(Y); free(a); free(T);
    }
    free(H); free(slot);
    free(row_ptr);
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* Parity-labelled inputs (Sec. VI A-E :193-:240, Sec. VII C a-c, e :383-:469).                   */
/*                                                                                              */
/* A feature I_{n l m, p} carries an absolute parity label p = +-1 next to l.  Storage (reading   */
/* R19): slot 0 of the slot axis holds the natural-parity part p = (-1)^l, slot 1 the  */
/* opposite-parity part p = -(-1)^l -- for every l the same two numbers as the paper's (+1, -1)   */
/* slots, indexed relative to (-1)^l.  The output uses the same two slots (= the two sectors of   */
/* the natural-parity entry points).                                                            */
/*                                                                                              */
/* What is evaluated is Eq.(2) / Eq.(1) with the output parity p = p1 p2 (:29, :240; B7's         */
/* dispatch rule p = (-1)^{l1} p2, :647) applied TERM BY TERM: every non-zero (l1m1, l2m2 -> lm)  */
/* of the Gaunt table (l1+l2+l even, Category alpha, Cases A and C) and of the Q table (l1+l2+l   */
/* odd, Category beta, Cases B and D) is routed to the output slot that p = p1 p2 and l select.   */
/* Following Eq.(42)-(43), (45), (56) every run has independent CP weights; with the l-shared     */
/* weights of reading R5 a run is one (category, slots, output-l parity sigma) combination:       */
/*   message passing: run r = 4*cat + 2*s_out + tau, tau = 0 for sigma = +1 (even l), 1 for odd   */
/*     l; cat 0 = alpha, 1 = beta; s_out the output slot.  (p, sigma) of Eq.(44)-(45) is          */
/*     (s_out, tau) with p = (-1)^{s_out} sigma.  8 runs.                                        */
/*   on-site (VII C e): run r = 8*cat + 4*s1 + 2*s2 + tau over the slots of both factors: 16 runs */
/*     ("two pairs x two output sectors x two output-l parities" x {alpha, beta}, :469).          */
/* Nothing below hard-codes which source slot feeds which output slot: that is decided per term   */
/* from the parities, so Eq.(44), (45), (56) are consequences the tests can check.                */
/* ------------------------------------------------------------------------------------------ */
static int isqrt_floor(int i)
{
    int l = (int)floor(sqrt((double)i));
    while ((l + 1) * (l + 1) <= i) ++l;
    while (l * l > i) --l;
    return l;
}
static int sgn_pow(int k) { return (k & 1) ? -1 : 1; }

/* node_feats [nodes,2,N,L2]; edge_radial [E,8,C]; l1_weight [lmax+1] or NULL (an l1-dependent     */
/* factor on the edge side, used by the dispatch pin B7 :647 to restrict the edge to one degree);  */
/* W_node [8,C,N]; W_out [8,N,C]; out [n_recv or nodes, 2, N, Lo2].                                */
int oracle_message_parity(const double *node_feats, const int64_t *edge_index, const double *edge_vec,
                          const double *edge_radial, const double *l1_weight, const double *W_node,
                          const double *W_out, int lmax, int lmax_out, int N, int C, double *out,
                          int64_t nodes, int64_t E, const int64_t *recv_list, int64_t n_recv)
{
    enum { R = 8 };
    int L2 = (lmax + 1) * (lmax + 1), Lo2 = (lmax_out + 1) * (lmax_out + 1);
    const coupling_t *tab[2];
    tab[0] = get_coupling(lmax, lmax_out, 0);
    tab[1] = get_coupling(lmax, lmax_out, 1);
    if (!tab[0] || !tab[1]) return 2;
    int64_t *row_ptr = malloc((size_t)(nodes + 1) * sizeof(int64_t));
    int rc = oracle_segments(edge_index, E, nodes, row_ptr);
    if (rc) { free(row_ptr); return rc; }
    const int64_t *snd = edge_index;
    int64_t nr = recv_list ? n_recv : nodes;
    int64_t *slot = malloc((size_t)nodes * sizeof(int64_t));
    for (int64_t j = 0; j < nodes; ++j) slot[j] = -1;
    int64_t n_need = 0;
    for (int64_t r = 0; r < nr; ++r) {
        int64_t i = recv_list ? recv_list[r] : r;
        for (int64_t e = row_ptr[i]; e < row_ptr[i + 1]; ++e)
            if (slot[snd[e]] < 0) slot[snd[e]] = n_need++;
    }
    /* Eq.(47) for every run and both source slots: H[j][run][s_in][c][l2m2] */
    size_t hsz = (size_t)R * 2 * C * L2;
    double *H = malloc((size_t)(n_need > 0 ? n_need : 1) * hsz * sizeof(double));
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t j = 0; j < nodes; ++j) {
        if (slot[j] < 0) continue;
        for (int run = 0; run < R; ++run)
            for (int s = 0; s < 2; ++s) {
                const double *xj = node_feats + (j * 2 + s) * (int64_t)N * L2;
                double *hj = H + slot[j] * hsz + ((size_t)run * 2 + s) * C * L2;
                for (int c = 0; c < C; ++c)
                    for (int q = 0; q < L2; ++q) {
                        double acc = 0.0;
                        for (int n = 0; n < N; ++n) acc += W_node[((size_t)run * C + c) * N + n] * xj[n * L2 + q];
                        hj[c * L2 + q] = acc;
                    }
            }
    }
#pragma omp parallel
    {
        double *Y = malloc((size_t)L2 * sizeof(double));
        double *T = malloc((size_t)R * C * Lo2 * sizeof(double));
#pragma omp for schedule(dynamic, 1)
        for (int64_t r = 0; r < nr; ++r) {
            int64_t i = recv_list ? recv_list[r] : r;
            for (size_t k = 0; k < (size_t)R * C * Lo2; ++k) T[k] = 0.0;
            for (int64_t e = row_ptr[i]; e < row_ptr[i + 1]; ++e) {
                oracle_real_sh(lmax, edge_vec[3 * e], edge_vec[3 * e + 1], edge_vec[3 * e + 2], Y);
                if (l1_weight)
                    for (int q = 0; q < L2; ++q) Y[q] *= l1_weight[isqrt_floor(q)];
                for (int run = 0; run < R; ++run) {
                    int cat = run >> 2, s_out = (run >> 1) & 1, tau = run & 1;
                    const coupling_t *t = tab[cat];
                    for (int s_in = 0; s_in < 2; ++s_in) {
                        const double *hj = H + slot[snd[e]] * hsz + ((size_t)run * 2 + s_in) * C * L2;
                        for (int64_t k = 0; k < t->nnz; ++k) {
                            int l1 = isqrt_floor(t->i1[k]), l2 = isqrt_floor(t->i2[k]), l = isqrt_floor(t->io[k]);
                            int p1 = sgn_pow(l1);              /* edge feature R Y_{l1}: natural parity (:370)      */
                            int p2 = sgn_pow(s_in) * sgn_pow(l2); /* parity label of the source slot               */
                            int p = p1 * p2;                   /* output parity, Eq.(2) / B7 (:647)                 */
                            int so = (p == sgn_pow(l)) ? 0 : 1;
                            if (so != s_out || (l & 1) != tau) continue; /* not a term of this run (Eq.(54): (-1)^l = sigma) */
                            for (int c = 0; c < C; ++c)
                                T[((size_t)run * C + c) * Lo2 + t->io[k]] +=
                                    t->val[k] * edge_radial[(e * R + run) * (int64_t)C + c] * Y[t->i1[k]] *
                                    hj[(size_t)c * L2 + t->i2[k]];
                        }
                    }
                }
            }
            /* Eq.(55), (58), (59): channel projection per run, alpha + beta summed into the output slot */
            double *ob = out + r * 2 * (int64_t)N * Lo2;
            for (size_t k = 0; k < (size_t)2 * N * Lo2; ++k) ob[k] = 0.0;
            for (int run = 0; run < R; ++run) {
                int s_out = (run >> 1) & 1;
                for (int n = 0; n < N; ++n)
                    for (int q = 0; q < Lo2; ++q) {
                        double acc = 0.0;
                        for (int c = 0; c < C; ++c)
                            acc += W_out[((size_t)run * N + n) * C + c] * T[((size_t)run * C + c) * Lo2 + q];
                        ob[((size_t)s_out * N + n) * Lo2 + q] += acc;
                    }
            }
        }
        free(Y); free(T);
    }
    free(H); free(slot); free(row_ptr);
    return 0;
}

/* A, B [batch,2,N,L2]; W_a, W_b [16,C,N]; W_out [16,N,C]; out [batch,2,N,Lo2].                    */
int oracle_onsite_parity(const double *A, const double *B, const double *W_a, const double *W_b,
                         const double *W_out, int lmax, int lmax_out, int N, int C, double *out, int64_t batch)
{
    enum { R = 16 };
    int L2 = (lmax + 1) * (lmax + 1), Lo2 = (lmax_out + 1) * (lmax_out + 1);
    const coupling_t *tab[2];
    tab[0] = get_coupling(lmax, lmax_out, 0);
    tab[1] = get_coupling(lmax, lmax_out, 1);
    if (!tab[0] || !tab[1]) return 2;
#pragma omp parallel
    {
        double *Ha = malloc((size_t)C * L2 * sizeof(double));
        double *Hb = malloc((size_t)C * L2 * sizeof(double));
        double *T = malloc((size_t)2 * C * Lo2 * sizeof(double)); /* [output slot][c][lm] of one run */
#pragma omp for schedule(dynamic, 1)
        for (int64_t b = 0; b < batch; ++b) {
            double *ob = out + b * 2 * (int64_t)N * Lo2;
            for (size_t k = 0; k < (size_t)2 * N * Lo2; ++k) ob[k] = 0.0;
            for (int run = 0; run < R; ++run) {
                int cat = run >> 3, s1 = (run >> 2) & 1, s2 = (run >> 1) & 1, tau = run & 1;
                const double *Ab = A + (b * 2 + s1) * (int64_t)N * L2, *Bb = B + (b * 2 + s2) * (int64_t)N * L2;
                for (int c = 0; c < C; ++c)
                    for (int q = 0; q < L2; ++q) {
                        double sa = 0.0, sb = 0.0;
                        for (int n = 0; n < N; ++n) {
                            sa += W_a[((size_t)run * C + c) * N + n] * Ab[n * L2 + q];
                            sb += W_b[((size_t)run * C + c) * N + n] * Bb[n * L2 + q];
                        }
                        Ha[c * L2 + q] = sa;
                        Hb[c * L2 + q] = sb;
                    }
                for (size_t k = 0; k < (size_t)2 * C * Lo2; ++k) T[k] = 0.0;
                const coupling_t *t = tab[cat];
                for (int64_t k = 0; k < t->nnz; ++k) {
                    int l1 = isqrt_floor(t->i1[k]), l2 = isqrt_floor(t->i2[k]), l = isqrt_floor(t->io[k]);
                    int p1 = sgn_pow(s1) * sgn_pow(l1), p2 = sgn_pow(s2) * sgn_pow(l2);
                    int p = p1 * p2;                        /* Eq.(1): output parity p = p1 p2 (:29)        */
                    int so = (p == sgn_pow(l)) ? 0 : 1;
                    if ((l & 1) != tau) continue;           /* this run feeds (-1)^l = sigma only           */
                    for (int c = 0; c < C; ++c)
                        T[((size_t)so * C + c) * Lo2 + t->io[k]] +=
                            t->val[k] * Ha[(size_t)c * L2 + t->i1[k]] * Hb[(size_t)c * L2 + t->i2[k]];
                }
                for (int so = 0; so < 2; ++so)
                    for (int n = 0; n < N; ++n)
                        for (int q = 0; q < Lo2; ++q) {
                            double acc = 0.0;
                            for (int c = 0; c < C; ++c)
                                acc += W_out[((size_t)run * N + n) * C + c] * T[((size_t)so * C + c) * Lo2 + q];
                            ob[((size_t)so * N + n) * Lo2 + q] += acc;
                        }
            }
        }
        free(Ha); free(Hb); free(T);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* l-dependent CP weights (the paper's own parameterisation: c_{cnl} in Eq.(35) :322 and Eq.(47)  */
/* :398, lambda_c^{(nl)} in Eq.(41) :346 and Eq.(55) :427; reading R5 made them l-shared for the  */
/* BASELINE configs).  W_a, W_b, W_node: [lmax+1, C, N]; W_out: [lmax_out+1, N, C]:               */
/*   H[c,lm] = sum_n W[l][c,n] A[n,lm]          out[s,n,lm] = sum_{c in s} W_out[l][n,c] T[c,lm]  */
/* The radial factor of the edge stays l1-shared (reading R12).  Everything else as oracle_onsite */
/* / oracle_message.                                                                            */
/* ------------------------------------------------------------------------------------------ */
int oracle_onsite_lw(const double *A, const double *B, const double *W_a, const double *W_b,
                     const double *W_out, int lmax, int lmax_out, int N, int C, const uint8_t *parity_mask,
                     double *out, int64_t batch)
{
    int L2 = (lmax + 1) * (lmax + 1), Lo2 = (lmax_out + 1) * (lmax_out + 1);
    const coupling_t *tab[2];
    tab[0] = get_coupling(lmax, lmax_out, 0);
    tab[1] = get_coupling(lmax, lmax_out, 1);
    if (!tab[0] || !tab[1]) return 2;
#pragma omp parallel
    {
        double *Ha = malloc((size_t)C * L2 * sizeof(double));
        double *Hb = malloc((size_t)C * L2 * sizeof(double));
        double *T = malloc((size_t)C * Lo2 * sizeof(double));
#pragma omp for schedule(dynamic, 1)
        for (int64_t b = 0; b < batch; ++b) {
            const double *Ab = A + b * (int64_t)N * L2, *Bb = B + b * (int64_t)N * L2;
            for (int c = 0; c < C; ++c)
                for (int i = 0; i < L2; ++i) {
                    int l = isqrt_floor(i);
                    double sa = 0.0, sb = 0.0;
                    for (int n = 0; n < N; ++n) {
                        sa += W_a[((size_t)l * C + c) * N + n] * Ab[n * L2 + i];
                        sb += W_b[((size_t)l * C + c) * N + n] * Bb[n * L2 + i];
                    }
                    Ha[c * L2 + i] = sa;
                    Hb[c * L2 + i] = sb;
                }
            for (int c = 0; c < C; ++c) {
                const coupling_t *t = tab[parity_mask[c] ? 1 : 0];
                double *Tc = T + (size_t)c * Lo2;
                for (int i = 0; i < Lo2; ++i) Tc[i] = 0.0;
                for (int64_t k = 0; k < t->nnz; ++k)
                    Tc[t->io[k]] += t->val[k] * Ha[(size_t)c * L2 + t->i1[k]] * Hb[(size_t)c * L2 + t->i2[k]];
            }
            double *ob = out + b * 2 * (int64_t)N * Lo2;
            for (int s = 0; s < 2; ++s)
                for (int n = 0; n < N; ++n)
                    for (int i = 0; i < Lo2; ++i) {
                        int l = isqrt_floor(i);
                        double acc = 0.0;
                        for (int c = 0; c < C; ++c)
                            if ((parity_mask[c] ? 1 : 0) == s)
                                acc += W_out[((size_t)l * N + n) * C + c] * T[(size_t)c * Lo2 + i];
                        ob[((size_t)s * N + n) * Lo2 + i] = acc;
                    }
        }
        free(Ha); free(Hb); free(T);
    }
    return 0;
}

/* radial_l1 = 0: edge_radial [E,C] (l1-shared, reading R12); radial_l1 = 1: edge_radial [E,C,lmax+1], the paper's  */
/* R~_{jicl1} of Eq.(46) (:396): a[e,c,l1m1] = edge_radial[e,c,l1] Y_{l1m1}(r_hat_e) (Eq.(48) :402).                   */
static int message_lw_impl(const double *node_feats, const int64_t *edge_index, const double *edge_vec,
                           const double *edge_radial, int radial_l1, const double *W_node, const double *W_out,
                           int lmax, int lmax_out, int N, int C, const uint8_t *parity_mask, double *out,
                           int64_t nodes, int64_t E)
{
    int L2 = (lmax + 1) * (lmax + 1), Lo2 = (lmax_out + 1) * (lmax_out + 1);
    const coupling_t *tab[2];
    tab[0] = get_coupling(lmax, lmax_out, 0);
    tab[1] = get_coupling(lmax, lmax_out, 1);
    if (!tab[0] || !tab[1]) return 2;
    int64_t *row_ptr = malloc((size_t)(nodes + 1) * sizeof(int64_t));
    int rc = oracle_segments(edge_index, E, nodes, row_ptr);
    if (rc) { free(row_ptr); return rc; }
    const int64_t *snd = edge_index;
    double *H = malloc((size_t)(nodes > 0 ? nodes : 1) * C * L2 * sizeof(double));
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t j = 0; j < nodes; ++j) {
        const double *xj = node_feats + j * (int64_t)N * L2;
        double *hj = H + j * (int64_t)C * L2;
        for (int c = 0; c < C; ++c)
            for (int q = 0; q < L2; ++q) {
                int l = isqrt_floor(q);
                double s = 0.0;
                for (int n = 0; n < N; ++n) s += W_node[((size_t)l * C + c) * N + n] * xj[n * L2 + q];
                hj[c * L2 + q] = s;
            }
    }
#pragma omp parallel
    {
        double *Y = malloc((size_t)L2 * sizeof(double));
        double *T = malloc((size_t)C * Lo2 * sizeof(double));
#pragma omp for schedule(dynamic, 1)
        for (int64_t i = 0; i < nodes; ++i) {
            for (size_t k = 0; k < (size_t)C * Lo2; ++k) T[k] = 0.0;
            for (int64_t e = row_ptr[i]; e < row_ptr[i + 1]; ++e) {
                const double *hj = H + snd[e] * (int64_t)C * L2;
                oracle_real_sh(lmax, edge_vec[3 * e], edge_vec[3 * e + 1], edge_vec[3 * e + 2], Y);
                for (int c = 0; c < C; ++c) {
                    const coupling_t *t = tab[parity_mask[c] ? 1 : 0];
                    for (int64_t k = 0; k < t->nnz; ++k) {
                        double rad = radial_l1 ? edge_radial[(e * (int64_t)C + c) * (lmax + 1) + isqrt_floor(t->i1[k])]
                                               : edge_radial[e * (int64_t)C + c];
                        T[(size_t)c * Lo2 + t->io[k]] += t->val[k] * rad * Y[t->i1[k]] * hj[(size_t)c * L2 + t->i2[k]];
                    }
                }
            }
            double *ob = out + i * 2 * (int64_t)N * Lo2;
            for (int s = 0; s < 2; ++s)
                for (int n = 0; n < N; ++n)
                    for (int q = 0; q < Lo2; ++q) {
                        int l = isqrt_floor(q);
                        double acc = 0.0;
                        for (int c = 0; c < C; ++c)
                            if ((parity_mask[c] ? 1 : 0) == s)
                                acc += W_out[((size_t)l * N + n) * C + c] * T[(size_t)c * Lo2 + q];
                        ob[((size_t)s * N + n) * Lo2 + q] = acc;
                    }
        }
        free(Y); free(T);
    }
    free(H); free(row_ptr);
    return 0;
}

int oracle_message_lw(const double *node_feats, const int64_t *edge_index, const double *edge_vec,
                      const double *edge_radial, const double *W_node, const double *W_out, int lmax,
                      int lmax_out, int N, int C, const uint8_t *parity_mask, double *out, int64_t nodes,
                      int64_t E)
{
    return message_lw_impl(node_feats, edge_index, edge_vec, edge_radial, 0, W_node, W_out, lmax, lmax_out, N, C,
                           parity_mask, out, nodes, E);
}

/* The message-passing coupling in the paper's full parameterisation: l-dependent c_{cnl}, lambda_c^{(nl)} and the   */
/* l1-dependent radial factor R~_{jicl1} (Eq.(46)-(48) :396-:402).  edge_radial [E, C, lmax+1].                        */
int oracle_message_lwr(const double *node_feats, const int64_t *edge_index, const double *edge_vec,
                       const double *edge_radial, const double *W_node, const double *W_out, int lmax,
                       int lmax_out, int N, int C, const uint8_t *parity_mask, double *out, int64_t nodes,
                       int64_t E)
{
    return message_lw_impl(node_feats, edge_index, edge_vec, edge_radial, 1, W_node, W_out, lmax, lmax_out, N, C,
                           parity_mask, out, nodes, E);
}

/* ------------------------------------------------------------------------------------------ */
/* nu-body on-site product (end of Sec. VI): "The grid pointwise product extends */
/* to nu-body features through additional pointwise multiplications on the grid followed by a  */
/* single inverse transform".  What that reaches exactly is the plain definition                */
/*   T[c,lm] = int prod_{s=1..nu} A~(s)_c(Omega) Y_lm(Omega) dOmega,  A~(s)_c = sum_i H(s)[c,i] Y_i, */
/*   H(s)[c,:] = W_in[s][c,:] . X[s][b]   (Eq.(35) :322 per factor),                            */
/*   out[b,n,lm] = sum_c W_out[n,c] T[c,lm]   (Eq.(41) :346; a product of natural-parity fields  */
/*   has natural parity: one sector).                                                           */
/* Written out with the real Gaunt tensor Gr (Eq.(4)-(5)) applied nu-1 times, the intermediate   */
/* products kept at their FULL band k*lmax (a product of k fields of band lmax has band k*lmax;  */
/* truncating it earlier would change the result):                                               */
/*   P_1 = H(1);  P_k[i] = sum_{a,b} Gr(a,b;i) P_{k-1}[a] H(k)[b],  band k*lmax;                 */
/*   T = P_nu restricted to l <= lmax_out.                                                       */
/* Nothing here touches a quadrature grid.  Reading R23: l-shared weights, rank       */
/* channels of the pointwise (even) kind only -- the curl pairing is bilinear and the paper       */
/* gives no nu-body form of it.  Layouts: X [nu,batch,N,(lmax+1)^2]; W_in [nu,C,N]; W_out [N,C];  */
/* out [batch,N,(lmax_out+1)^2].                                                                  */
/* ------------------------------------------------------------------------------------------ */
int oracle_onsite_nbody(const double *X, const double *W_in, const double *W_out, int nu, int lmax, int lmax_out,
                        int N, int C, double *out, int64_t batch)
{
    if (nu < 1 || nu > 8 || lmax < 0 || lmax_out < 0 || lmax_out > nu * lmax) return 1;
    int L2 = (lmax + 1) * (lmax + 1), Lo2 = (lmax_out + 1) * (lmax_out + 1);
    /* step k (2..nu): left band (k-1)*lmax, right band lmax, output band k*lmax (last step: lmax_out) */
    const coupling_t *tab[9];
    int lin[9], lout[9];
    for (int k = 2; k <= nu; ++k) {
        lin[k] = (k - 1) * lmax;
        lout[k] = (k == nu) ? lmax_out : k * lmax;
        tab[k] = get_coupling(lin[k], lout[k], 0);
        if (!tab[k]) return 2;
    }
    int Pmax = (nu * lmax + 1) * (nu * lmax + 1);
#pragma omp parallel
    {
        double *H = malloc((size_t)nu * C * L2 * sizeof(double));
        double *P = malloc((size_t)Pmax * sizeof(double));
        double *Pn = malloc((size_t)Pmax * sizeof(double));
        double *T = malloc((size_t)C * Lo2 * sizeof(double));
#pragma omp for schedule(dynamic, 1)
        for (int64_t b = 0; b < batch; ++b) {
            for (int s = 0; s < nu; ++s) {
                const double *Xb = X + ((int64_t)s * batch + b) * N * L2;
                const double *W = W_in + (size_t)s * C * N;
                for (int c = 0; c < C; ++c)
                    for (int i = 0; i < L2; ++i) {
                        double acc = 0.0;
                        for (int n = 0; n < N; ++n) acc += W[c * N + n] * Xb[n * L2 + i];
                        H[((size_t)s * C + c) * L2 + i] = acc;
                    }
            }
            for (int c = 0; c < C; ++c) {
                for (int i = 0; i < Pmax; ++i) P[i] = 0.0;
                for (int i = 0; i < L2; ++i) P[i] = H[(size_t)c * L2 + i];
                if (nu == 1) { /* single field: T = H restricted to lmax_out (lmax_out <= lmax) */ }
                for (int k = 2; k <= nu; ++k) {
                    const coupling_t *t = tab[k];
                    const double *h = H + ((size_t)(k - 1) * C + c) * L2;
                    int no = (lout[k] + 1) * (lout[k] + 1);
                    for (int i = 0; i < Pmax; ++i) Pn[i] = 0.0;
                    for (int64_t q = 0; q < t->nnz; ++q)
                        if (t->i2[q] < L2) /* factor k has band lmax; the table covers band (k-1)*lmax on both sides */
                            Pn[t->io[q]] += t->val[q] * P[t->i1[q]] * h[t->i2[q]];
                    for (int i = 0; i < Pmax; ++i) P[i] = (i < no) ? Pn[i] : 0.0;
                }
                for (int i = 0; i < Lo2; ++i) T[(size_t)c * Lo2 + i] = P[i];
            }
            double *ob = out + b * (int64_t)N * Lo2;
            for (int n = 0; n < N; ++n)
                for (int i = 0; i < Lo2; ++i) {
                    double acc = 0.0;
                    for (int c = 0; c < C; ++c) acc += W_out[n * C + c] * T[(size_t)c * Lo2 + i];
                    ob[(size_t)n * Lo2 + i] = acc;
                }
        }
        free(H); free(P); free(Pn); free(T);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* Two feature fields, Eq.(28) (Sec. VII C f :471): the edge side is a general      */
/* feature field I^(E)[e,n1,l1m1] that no longer factors as R.Y, the node side the sender's       */
/* feature I^(N)[j,n2,l2m2].  With the CP factorisation (Eq.(3) :39; "an explicit radial          */
/* contraction ... on the edge side, replacing R~ by an analogue of Eq.(47)", :471):              */
/*   a[e,c,:]  = W_edge[c,:] . edge_feats[e]                 (factor 1, analogue of Eq.(47))      */
/*   H[j,c,:]  = W_node[c,:] . node_feats[j]                 (factor 2, Eq.(47) :398)             */
/*   T[i,c,lm] = sum_{e: recv(e)=i} sum coef(i1,i2;lm) a[e,c,i1] H[send(e),c,i2]                  */
/*               coef = Gr (mask 0, Category alpha) or Qr (mask 1, Category beta, Eq.(57) :443)   */
/*   out[i,s,n,lm] = sum_{c: mask[c]=s} W_out[n,c] T[i,c,lm]                                      */
/* Reading R21: natural-parity slots on both fields (the (p1,p2) slot dispatch of     */
/* :471 is a routing layer over this coupling, as in oracle_*_parity), l-shared weights (R5).     */
/* Layouts: node_feats [nodes,N,L2]; edge_feats [E,Ne,L2]; W_edge [C,Ne]; W_node [C,N];           */
/* W_out [N,C]; out [nodes,2,N,Lo2].                                                              */
/* ------------------------------------------------------------------------------------------ */
/* lw = 1: l-dependent weights (the paper's own parameterisation, Eq.(35) :322, (41) :346, (47) :398, (55) :427):  */
/* W_edge [lmax+1,C,Ne], W_node [lmax+1,C,N] act on the coefficients of their degree l, W_out [lmax_out+1,N,C] on   */
/* the output coefficients of its degree.                                                                          */
static int message_field_impl(const double *node_feats, const int64_t *edge_index /* [2,E] */, const double *edge_feats,
                              const double *W_edge, const double *W_node, const double *W_out, int lmax, int lmax_out,
                              int N, int Ne, int C, const uint8_t *parity_mask, double *out, int64_t nodes, int64_t E,
                              int lw)
{
    int L2 = (lmax + 1) * (lmax + 1), Lo2 = (lmax_out + 1) * (lmax_out + 1);
    const coupling_t *tab[2];
    tab[0] = get_coupling(lmax, lmax_out, 0);
    tab[1] = get_coupling(lmax, lmax_out, 1);
    if (!tab[0] || !tab[1]) return 2;
    int64_t *row_ptr = malloc((size_t)(nodes + 1) * sizeof(int64_t));
    int rc = oracle_segments(edge_index, E, nodes, row_ptr);
    if (rc) { free(row_ptr); return rc; }
    const int64_t *snd = edge_index;
#pragma omp parallel
    {
        double *a = malloc((size_t)C * L2 * sizeof(double));
        double *h = malloc((size_t)C * L2 * sizeof(double));
        double *T = malloc((size_t)C * Lo2 * sizeof(double));
#pragma omp for schedule(dynamic, 1)
        for (int64_t i = 0; i < nodes; ++i) {
            for (size_t k = 0; k < (size_t)C * Lo2; ++k) T[k] = 0.0;
            for (int64_t e = row_ptr[i]; e < row_ptr[i + 1]; ++e) {
                const double *xe = edge_feats + e * (int64_t)Ne * L2;
                const double *xj = node_feats + snd[e] * (int64_t)N * L2;
                for (int c = 0; c < C; ++c)
                    for (int q = 0; q < L2; ++q) {
                        const int l = lw ? isqrt_floor(q) : 0;
                        const double *We = W_edge + (size_t)l * C * Ne, *Wn = W_node + (size_t)l * C * N;
                        double sa = 0.0, sh = 0.0;
                        for (int n = 0; n < Ne; ++n) sa += We[c * Ne + n] * xe[n * L2 + q];
                        for (int n = 0; n < N; ++n) sh += Wn[c * N + n] * xj[n * L2 + q];
                        a[c * L2 + q] = sa;
                        h[c * L2 + q] = sh;
                    }
                for (int c = 0; c < C; ++c) {
                    const coupling_t *t = tab[parity_mask[c] ? 1 : 0];
                    double *Tc = T + (size_t)c * Lo2;
                    const double *ac = a + (size_t)c * L2, *hc = h + (size_t)c * L2;
                    for (int64_t k = 0; k < t->nnz; ++k)
                        Tc[t->io[k]] += t->val[k] * ac[t->i1[k]] * hc[t->i2[k]];
                }
            }
            double *ob = out + i * 2 * (int64_t)N * Lo2;
            for (int s = 0; s < 2; ++s)
                for (int n = 0; n < N; ++n)
                    for (int q = 0; q < Lo2; ++q) {
                        const double *Wo = W_out + (size_t)(lw ? isqrt_floor(q) : 0) * N * C;
                        double acc = 0.0;
                        for (int c = 0; c < C; ++c)
                            if ((parity_mask[c] ? 1 : 0) == s) acc += Wo[n * C + c] * T[(size_t)c * Lo2 + q];
                        ob[((size_t)s * N + n) * Lo2 + q] = acc;
                    }
        }
        free(a); free(h); free(T);
    }
    free(row_ptr);
    return 0;
}

int oracle_message_field(const double *node_feats, const int64_t *edge_index, const double *edge_feats,
                         const double *W_edge, const double *W_node, const double *W_out, int lmax, int lmax_out,
                         int N, int Ne, int C, const uint8_t *parity_mask, double *out, int64_t nodes, int64_t E)
{
    return message_field_impl(node_feats, edge_index, edge_feats, W_edge, W_node, W_out, lmax, lmax_out, N, Ne, C,
                              parity_mask, out, nodes, E, 0);
}

int oracle_message_field_lw(const double *node_feats, const int64_t *edge_index, const double *edge_feats,
                            const double *W_edge, const double *W_node, const double *W_out, int lmax, int lmax_out,
                            int N, int Ne, int C, const uint8_t *parity_mask, double *out, int64_t nodes, int64_t E)
{
    return message_field_impl(node_feats, edge_index, edge_feats, W_edge, W_node, W_out, lmax, lmax_out, N, Ne, C,
                              parity_mask, out, nodes, E, 1);
}

/* ------------------------------------------------------------------------------------------ */
/* Two parity-bearing fields, Eq.(28) with the parity labels of both fields        */
/* (Sec. VI E :232-:240; Sec. VII C f :471).  Slot axes as in oracle_onsite_parity (R19): */
/* slot 0 = natural parity (-1)^l, slot 1 = opposite parity.  Runs r = 8 cat + 4 s1 + 2 s2 + tau    */
/* (R20): category cat (0: Gaunt, 1: curl), slot s1 of the edge field (factor 1, R10), slot s2 of   */
/* the node field, output-degree parity tau.  Every non-zero coupling term is routed by p = p1 p2   */
/* (:236 "The output parity is p = p1 p2") to the output slot whose label it carries.               */
/*   edge_feats [E][2][Ne][L2], node_feats [nodes][2][N][L2],                                       */
/*   W_edge [16][C][Ne], W_node [16][C][N], W_out [16][N][C], out [nodes][2][N][Lo2].               */
/* ------------------------------------------------------------------------------------------ */
int oracle_message_field_parity(const double *node_feats, const int64_t *edge_index, const double *edge_feats,
                                const double *W_edge, const double *W_node, const double *W_out, int lmax,
                                int lmax_out, int N, int Ne, int C, double *out, int64_t nodes, int64_t E)
{
    enum { R = 16 };
    int L2 = (lmax + 1) * (lmax + 1), Lo2 = (lmax_out + 1) * (lmax_out + 1);
    const coupling_t *tab[2];
    tab[0] = get_coupling(lmax, lmax_out, 0);
    tab[1] = get_coupling(lmax, lmax_out, 1);
    if (!tab[0] || !tab[1]) return 2;
    int64_t *row_ptr = malloc((size_t)(nodes + 1) * sizeof(int64_t));
    int rc = oracle_segments(edge_index, E, nodes, row_ptr);
    if (rc) { free(row_ptr); return rc; }
    const int64_t *snd = edge_index;
#pragma omp parallel
    {
        double *a = malloc((size_t)C * L2 * sizeof(double));
        double *h = malloc((size_t)C * L2 * sizeof(double));
        double *T = malloc((size_t)2 * C * Lo2 * sizeof(double)); /* [output slot][c][lm] of one run */
#pragma omp for schedule(dynamic, 1)
        for (int64_t i = 0; i < nodes; ++i) {
            double *ob = out + i * 2 * (int64_t)N * Lo2;
            for (size_t k = 0; k < (size_t)2 * N * Lo2; ++k) ob[k] = 0.0;
            for (int run = 0; run < R; ++run) {
                int cat = run >> 3, s1 = (run >> 2) & 1, s2 = (run >> 1) & 1, tau = run & 1;
                const coupling_t *t = tab[cat];
                for (size_t k = 0; k < (size_t)2 * C * Lo2; ++k) T[k] = 0.0;
                for (int64_t e = row_ptr[i]; e < row_ptr[i + 1]; ++e) {
                    const double *xe = edge_feats + (e * 2 + s1) * (int64_t)Ne * L2;
                    const double *xj = node_feats + (snd[e] * 2 + s2) * (int64_t)N * L2;
                    for (int c = 0; c < C; ++c)
                        for (int q = 0; q < L2; ++q) {
                            double sa = 0.0, sh = 0.0;
                            for (int n = 0; n < Ne; ++n) sa += W_edge[((size_t)run * C + c) * Ne + n] * xe[n * L2 + q];
                            for (int n = 0; n < N; ++n) sh += W_node[((size_t)run * C + c) * N + n] * xj[n * L2 + q];
                            a[c * L2 + q] = sa;
                            h[c * L2 + q] = sh;
                        }
                    for (int64_t k = 0; k < t->nnz; ++k) {
                        int l1 = isqrt_floor(t->i1[k]), l2 = isqrt_floor(t->i2[k]), l = isqrt_floor(t->io[k]);
                        int p1 = sgn_pow(s1) * sgn_pow(l1), p2 = sgn_pow(s2) * sgn_pow(l2);
                        int p = p1 * p2;                        /* Eq.(28): output parity p = p1 p2 (:236)      */
                        int so = (p == sgn_pow(l)) ? 0 : 1;
                        if ((l & 1) != tau) continue;           /* this run feeds (-1)^l = sigma only (Eq.(54)) */
                        for (int c = 0; c < C; ++c)
                            T[((size_t)so * C + c) * Lo2 + t->io[k]] +=
                                t->val[k] * a[(size_t)c * L2 + t->i1[k]] * h[(size_t)c * L2 + t->i2[k]];
                    }
                }
                for (int so = 0; so < 2; ++so)
                    for (int n = 0; n < N; ++n)
                        for (int q = 0; q < Lo2; ++q) {
                            double acc = 0.0;
                            for (int c = 0; c < C; ++c)
                                acc += W_out[((size_t)run * N + n) * C + c] * T[((size_t)so * C + c) * Lo2 + q];
                            ob[((size_t)so * N + n) * Lo2 + q] += acc;
                        }
            }
        }
        free(a); free(h); free(T);
    }
    free(row_ptr);
    return 0;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
