// sht.cuh -- device building blocks of the structured-grid transforms (SURVEY.md 8(a) rows S2a, S2b,
// S3, S4a, S4b / M2, M5), shared by the fused on-site kernel and the message-passing kernels.
//
// Coefficient rows.  For one grid row u the azimuthal coefficient vector of a field is stored as
// M = 2*LB+1 "rows": row m (0..LB) multiplies the cosine functions q_{v,+m}, row LB+a (a = 1..LB)
// multiplies the sine functions q_{v,-a} of Eq.(C2).
// F arrays in shared memory are [M][J] with J = NC*U and j = col*U + u the fastest index, so the
// thread that owns (col,u) reads a conflict-free column.
//
// Folding: Legendre sums are split into the parts even / odd under
// x -> -x, so one table row serves the node pair (u', U-1-u'); the real DFT is split into its cosine
// and sine parts, so one table row serves the azimuth pair (v', V-v').
#pragma once

#include "common.cuh"

namespace cgtp {

// ------------------------------------------------------------------------------- TMA / mbarrier
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t phase)
{
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(phase)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t phase)
{
    while (!mbar_try_wait(bar, phase)) {
    }
}
// 1-D bulk copy global -> shared through the TMA engine (cp.async.bulk); bytes % 16 == 0, both
// addresses 16-byte aligned.  Completion is signalled on `bar` (complete_tx).
__device__ __forceinline__ void tma_load_1d(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// 1-D bulk copy shared -> global.
__device__ __forceinline__ void tma_store_1d(void* dst_gmem, const void* src_smem, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst_gmem), "r"(smem_u32(src_smem)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void tma_store_commit_wait()
{
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// The largest single bulk copy we issue (the tx-count field of an mbarrier is 20 bits).
constexpr uint32_t kTmaChunk = 1u << 16;

// Thread 0 issues the copies for [src, src+bytes) in chunks and arms the barrier with the total.
__device__ __forceinline__ void tma_load_span(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar)
{
    uint32_t off = 0;
    while (off < bytes) {
        uint32_t n = bytes - off < kTmaChunk ? bytes - off : kTmaChunk;
        tma_load_1d((char*)dst_smem + off, (const char*)src_gmem + off, n, bar);
        off += n;
    }
}

// ------------------------------------------------------------------------------ Legendre synthesis
// One destination of a Legendre pass: F rows of one field, with a sign.
struct LegDst {
    float* F;    // [M][J]
    float sign;  // multiplies everything written
};

// Rows S2a / M2 (Eq.(36), Eq.(49) :404; derivative passes :445).
// Work item = (column, |m|).  For NIN inputs (H of factor 1 and 2) and the tables of this parity:
//   ODD == false: value table PT                      -> dst[in][0]
//   ODD == true : d_theta table DT                    -> dst[in][0]
//                 (1/sin) d_phi table ST, cos<->sin swap of PAPER.md:679 -> dst[in][1]
// Hs: [NIN][NC][L2p] projected coefficients in shared memory.
template <int LB, bool ODD, int NIN, int UB>
__device__ __forceinline__ void legendre_synthesis(const float* __restrict__ tab0, const float* __restrict__ tab1,
                                                   const float* __restrict__ Hs, int h_in_stride, int L2p,
                                                   const LegDst (&dst)[NIN][2], int NC, int lmax, int U, int Uh,
                                                   int NTRI, int J)
{
    constexpr int NTAB = ODD ? 2 : 1;
    const int items = NC * (lmax + 1);
    for (int item = threadIdx.x; item < items; item += blockDim.x) {
        const int col = item / (lmax + 1);
        const int mm = item - col * (lmax + 1);
        const float* hcol = Hs + (size_t)col * L2p;
        for (int u0 = 0; u0 < Uh; u0 += UB) {
            // acc[in][tab][sgn(+m,-m)][parity of l-m][ub]
            float acc[NIN][NTAB][2][2][UB];
#pragma unroll
            for (int a = 0; a < NIN; ++a)
#pragma unroll
                for (int b = 0; b < NTAB; ++b)
#pragma unroll
                    for (int c = 0; c < 2; ++c)
#pragma unroll
                        for (int d = 0; d < 2; ++d)
#pragma unroll
                            for (int e = 0; e < UB; ++e) acc[a][b][c][d][e] = 0.f;

            for (int l = mm; l <= lmax; l += 2) {
#pragma unroll
                for (int par = 0; par < 2; ++par) {
                    const int ll = l + par;
                    if (ll > lmax) break;
                    const int t = tri_index(ll, mm);
                    float h[NIN][2];
#pragma unroll
                    for (int a = 0; a < NIN; ++a) {
                        h[a][0] = hcol[a * h_in_stride + ll * ll + ll + mm];
                        h[a][1] = hcol[a * h_in_stride + ll * ll + ll - mm];
                    }
#pragma unroll
                    for (int e = 0; e < UB; ++e) {
                        if (u0 + e < Uh) {
                            const float p0 = tab0[(u0 + e) * NTRI + t];
#pragma unroll
                            for (int a = 0; a < NIN; ++a) {
                                acc[a][0][0][par][e] = fmaf(p0, h[a][0], acc[a][0][0][par][e]);
                                acc[a][0][1][par][e] = fmaf(p0, h[a][1], acc[a][0][1][par][e]);
                            }
                            if (ODD) {
                                const float p1 = tab1[(u0 + e) * NTRI + t];
#pragma unroll
                                for (int a = 0; a < NIN; ++a) {
                                    acc[a][NTAB - 1][0][par][e] = fmaf(p1, h[a][0], acc[a][NTAB - 1][0][par][e]);
                                    acc[a][NTAB - 1][1][par][e] = fmaf(p1, h[a][1], acc[a][NTAB - 1][1][par][e]);
                                }
                            }
                        }
                    }
                }
            }
            // scatter to the F rows of this |m|: north node u', south node U-1-u'
#pragma unroll
            for (int e = 0; e < UB; ++e) {
                const int up = u0 + e;
                if (up >= Uh) break;
                const int jn = col * U + up, js = col * U + (U - 1 - up);
#pragma unroll
                for (int a = 0; a < NIN; ++a) {
                    if (!ODD) {
                        // P~(-x) = (-1)^(l+m) P~(x): even part symmetric, odd part antisymmetric
                        const float s = dst[a][0].sign;
                        float* F = dst[a][0].F;
                        const float ep = acc[a][0][0][0][e], op = acc[a][0][0][1][e];
                        F[mm * J + jn] = s * (ep + op);
                        F[mm * J + js] = s * (ep - op);
                        if (mm > 0) {
                            const float en = acc[a][0][1][0][e], on = acc[a][0][1][1][e];
                            F[(LB + mm) * J + jn] = s * (en + on);
                            F[(LB + mm) * J + js] = s * (en - on);
                        }
                    } else {
                        // d/dtheta flips the reflection parity: even-(l-m) part antisymmetric
                        {
                            const float s = dst[a][0].sign;
                            float* F = dst[a][0].F;
                            const float ep = acc[a][0][0][0][e], op = acc[a][0][0][1][e];
                            F[mm * J + jn] = s * (ep + op);
                            F[mm * J + js] = s * (op - ep);
                            if (mm > 0) {
                                const float en = acc[a][0][1][0][e], on = acc[a][0][1][1][e];
                                F[(LB + mm) * J + jn] = s * (en + on);
                                F[(LB + mm) * J + js] = s * (on - en);
                            }
                        }
                        // (1/sin) d_phi: cos row +m takes +m*(sine coefficient), sine row takes -m*(cosine coefficient);
                        // the factor m is inside the ST table.
                        {
                            const float s = dst[a][1].sign;
                            float* F = dst[a][1].F;
                            const float ep = acc[a][1][0][0][e], op = acc[a][1][0][1][e];  // from H[l,+m]
                            const float en = acc[a][1][1][0][e], on = acc[a][1][1][1][e];  // from H[l,-m]
                            if (mm == 0) {
                                F[jn] = 0.f;
                                F[js] = 0.f;
                            } else {
                                F[mm * J + jn] = s * (en + on);
                                F[mm * J + js] = s * (en - on);
                                F[(LB + mm) * J + jn] = -s * (ep + op);
                                F[(LB + mm) * J + js] = -s * (ep - op);
                            }
                        }
                    }
                }
            }
        }
    }
}

// Zero the F rows above lmax when the kernel band limit LB exceeds lmax (lmax_out > lmax).
template <int LB>
__device__ __forceinline__ void zero_high_rows(float* F, int lmax, int J)
{
    if (lmax >= LB) return;
    const int nrow = LB - lmax;
    for (int idx = threadIdx.x; idx < 2 * nrow * J; idx += blockDim.x) {
        const int r = idx / J, j = idx - r * J;
        const int row = (r < nrow) ? (lmax + 1 + r) : (LB + lmax + 1 + (r - nrow));
        F[row * J + j] = 0.f;
    }
}

// ------------------------------------------------------------------------------- Fourier stages
template <int LB>
__device__ __forceinline__ void load_q_row(const float* __restrict__ Q, int vp, float (&q)[round_up(LB + 1, 4)])
{
    constexpr int QSTR = round_up(LB + 1, 4);
    const float4* src = reinterpret_cast<const float4*>(Q + vp * QSTR);
#pragma unroll
    for (int i = 0; i < QSTR / 4; ++i) {
        float4 t = src[i];
        q[4 * i] = t.x; q[4 * i + 1] = t.y; q[4 * i + 2] = t.z; q[4 * i + 3] = t.w;
    }
}

// Rows S2b + S3 + S4a fused for one (term, column, u) (Eq.(37)-(39) PAPER.md:327-:339):
// forward real DFT of the two coefficient vectors, pointwise product, inverse real DFT, in registers.
// FA/FB: [M][J] shared; the result T[m] overwrites FA[.][j].
template <int LB>
__device__ __forceinline__ void dft_product_idft(float* FA, const float* FB, int J, int j,
                                                 const float* __restrict__ QC, const float* __restrict__ QS,
                                                 const float* __restrict__ WV, int Vh)
{
    constexpr int M = 2 * LB + 1;
    constexpr int QSTR = round_up(LB + 1, 4);
    float fa[M], fb[M], t[M];
#pragma unroll
    for (int r = 0; r < M; ++r) {
        fa[r] = FA[r * J + j];
        fb[r] = FB[r * J + j];
        t[r] = 0.f;
    }
    for (int vp = 0; vp < Vh; ++vp) {
        float qc[QSTR], qs[QSTR];
        load_q_row<LB>(QC, vp, qc);
        load_q_row<LB>(QS, vp, qs);
        float cea = 0.f, ceb = 0.f, soa = 0.f, sob = 0.f;
#pragma unroll
        for (int m = 0; m <= LB; ++m) {
            cea = fmaf(qc[m], fa[m], cea);
            ceb = fmaf(qc[m], fb[m], ceb);
        }
#pragma unroll
        for (int m = 1; m <= LB; ++m) {
            soa = fmaf(qs[m], fa[LB + m], soa);
            sob = fmaf(qs[m], fb[LB + m], sob);
        }
        const float s1 = (cea + soa) * (ceb + sob);  // grid point v'
        const float s2 = (cea - soa) * (ceb - sob);  // mirrored grid point V - v'
        const float w = WV[vp];
        const float sp = w * (s1 + s2), sm = w * (s1 - s2);
#pragma unroll
        for (int m = 0; m <= LB; ++m) t[m] = fmaf(qc[m], sp, t[m]);
#pragma unroll
        for (int m = 1; m <= LB; ++m) t[LB + m] = fmaf(qs[m], sm, t[LB + m]);
    }
#pragma unroll
    for (int r = 0; r < M; ++r) FA[r * J + j] = t[r];
}

// Row M2 (Eq.(51)): forward real DFT of one coefficient vector to V grid values.
// F: [M][J] shared; grow: V floats (row u of one grid field) in shared memory.
template <int LB>
__device__ __forceinline__ void dft_forward_row(const float* F, int J, int j, float* grow,
                                                const float* __restrict__ QC, const float* __restrict__ QS, int V,
                                                int Vh)
{
    constexpr int M = 2 * LB + 1;
    constexpr int QSTR = round_up(LB + 1, 4);
    float f[M];
#pragma unroll
    for (int r = 0; r < M; ++r) f[r] = F[r * J + j];
    for (int vp = 0; vp < Vh; ++vp) {
        float qc[QSTR], qs[QSTR];
        load_q_row<LB>(QC, vp, qc);
        load_q_row<LB>(QS, vp, qs);
        float ce = 0.f, so = 0.f;
#pragma unroll
        for (int m = 0; m <= LB; ++m) ce = fmaf(qc[m], f[m], ce);
#pragma unroll
        for (int m = 1; m <= LB; ++m) so = fmaf(qs[m], f[LB + m], so);
        grow[vp] = ce + so;
        if (vp > 0) grow[V - vp] = ce - so;  // self-mirrored v' = V/2 writes the same value twice (so = 0)
    }
}

// Row M5 first half (Eq.(53)): inverse real DFT of one grid row to coefficient rows.
// srow: V floats in shared memory; result written to T[.][j] ([M][J] shared).
template <int LB>
__device__ __forceinline__ void dft_inverse_row(const float* srow, float* T, int J, int j,
                                                const float* __restrict__ QC, const float* __restrict__ QS,
                                                const float* __restrict__ WV, int V, int Vh)
{
    constexpr int M = 2 * LB + 1;
    constexpr int QSTR = round_up(LB + 1, 4);
    float t[M];
#pragma unroll
    for (int r = 0; r < M; ++r) t[r] = 0.f;
    for (int vp = 0; vp < Vh; ++vp) {
        float qc[QSTR], qs[QSTR];
        load_q_row<LB>(QC, vp, qc);
        load_q_row<LB>(QS, vp, qs);
        const float s1 = srow[vp];
        const float s2 = srow[vp == 0 ? 0 : V - vp];
        const float w = WV[vp];
        const float sp = w * (s1 + s2), sm = w * (s1 - s2);
#pragma unroll
        for (int m = 0; m <= LB; ++m) t[m] = fmaf(qc[m], sp, t[m]);
#pragma unroll
        for (int m = 1; m <= LB; ++m) t[LB + m] = fmaf(qs[m], sm, t[LB + m]);
    }
#pragma unroll
    for (int r = 0; r < M; ++r) T[r * J + j] = t[r];
}

// The azimuthal tables of one plan as a kernel parameter (constant bank): the table index depends only on the loop counter,
// so the loads run on the uniform datapath (LDCU) and the FMAs take the value as a uniform-register operand -- no
// shared-memory wavefronts, where the broadcast 128-bit loads of the shared-memory form cost two each (measured:
// the shared-memory pipe, not the FMA pipe, bound the transforms).
template <int LB>
struct QParam {
    static constexpr int QSTR = round_up(LB + 1, 4);
    static constexpr int VHMAX = (3 * LB + 1) / 2 + 1;  // Vh of the bilinear grid at lmax = lmax_out = LB
    float qc[VHMAX * QSTR], qs[VHMAX * QSTR], wv[round_up(VHMAX, 4)];
};
template <int LB>
inline void fill_qparam(const Plan* p, QParam<LB>& q)
{
    for (int i = 0; i < p->Vh * p->QSTR; ++i) { q.qc[i] = p->hQC[i]; q.qs[i] = p->hQS[i]; }
    for (int i = 0; i < round_up(p->Vh, 4); ++i) q.wv[i] = p->hWV[i];
}

// dft_inverse_row with the tables read from a QParam kernel parameter.
template <int LB>
__device__ __forceinline__ void dft_inverse_row_p(const float* srow, float* T, int J, int j, const QParam<LB>& q, int V, int Vh)
{
    constexpr int M = 2 * LB + 1;
    constexpr int QSTR = QParam<LB>::QSTR;
    float t[M];
#pragma unroll
    for (int r = 0; r < M; ++r) t[r] = 0.f;
    // fully unrolled over the largest Vh of the band limit: every table index is a compile-time constant, so the table
    // values are constant-bank operands of the FMAs themselves (no load instruction at all)
#pragma unroll
    for (int vp = 0; vp < QParam<LB>::VHMAX; ++vp) {
        if (vp >= Vh) break;
        const float s1 = srow[vp];
        const float s2 = srow[vp == 0 ? 0 : V - vp];
        const float w = q.wv[vp];
        const float sp = w * (s1 + s2), sm = w * (s1 - s2);
#pragma unroll
        for (int m = 0; m <= LB; ++m) t[m] = fmaf(q.qc[vp * QSTR + m], sp, t[m]);
#pragma unroll
        for (int m = 1; m <= LB; ++m) t[LB + m] = fmaf(q.qs[vp * QSTR + m], sm, t[LB + m]);
    }
#pragma unroll
    for (int r = 0; r < M; ++r) T[r * J + j] = t[r];
}

// --------------------------------------------------------------------------- Legendre analysis
// Rows S4b / M5 second half (Eq.(40), Eq.(54) :422): Gauss-Legendre quadrature.
// T0 (+ T1 if not null): [M][J] shared, the azimuthal coefficients per grid row; WP: [Uh][NTRI] table
// (weights folded in, equator halved); out: global [NC][Lo2p].
// UHMAX: upper bound of Uh; the default is Uh for lmax = lmax_out = LB on the bilinear grid, the largest possible there.
template <int LB, int UHMAX = ((3 * LB + 2) / 2 + 1) / 2>
__device__ __forceinline__ void legendre_analysis(const float* T0, const float* T1, const float* __restrict__ WP,
                                                  float* __restrict__ out, int Lo2p, int NC, int lmax_out, int U,
                                                  int Uh, int NTRI, int J)
{
    const int items = NC * (lmax_out + 1);
    for (int item = threadIdx.x; item < items; item += blockDim.x) {
        const int col = item / (lmax_out + 1);
        const int mm = item - col * (lmax_out + 1);
        float tp[2][UHMAX], tm[2][UHMAX];
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const int row = (s == 0) ? mm : (LB + mm);
#pragma unroll
            for (int up = 0; up < UHMAX; ++up) {
                float n = 0.f, so = 0.f;
                if (up < Uh && !(s == 1 && mm == 0)) {
                    n = T0[row * J + col * U + up];
                    so = T0[row * J + col * U + (U - 1 - up)];
                    if (T1) {
                        n += T1[row * J + col * U + up];
                        so += T1[row * J + col * U + (U - 1 - up)];
                    }
                }
                tp[s][up] = n + so;
                tm[s][up] = n - so;
            }
        }
        float* ocol = out + (size_t)col * Lo2p;
        for (int l = mm; l <= lmax_out; l += 2) {
            const int t0 = tri_index(l, mm);
            float ap = 0.f, an = 0.f;
#pragma unroll
            for (int up = 0; up < UHMAX; ++up) {
                if (up < Uh) {
                    const float wp = WP[up * NTRI + t0];
                    ap = fmaf(wp, tp[0][up], ap);
                    an = fmaf(wp, tp[1][up], an);
                }
            }
            ocol[l * l + l + mm] = ap;
            if (mm > 0) ocol[l * l + l - mm] = an;
            if (l + 1 <= lmax_out) {
                const int t1 = tri_index(l + 1, mm);
                float bp = 0.f, bn = 0.f;
#pragma unroll
                for (int up = 0; up < UHMAX; ++up) {
                    if (up < Uh) {
                        const float wp = WP[up * NTRI + t1];
                        bp = fmaf(wp, tm[0][up], bp);
                        bn = fmaf(wp, tm[1][up], bn);
                    }
                }
                ocol[(l + 1) * (l + 1) + (l + 1) + mm] = bp;
                if (mm > 0) ocol[(l + 1) * (l + 1) + (l + 1) - mm] = bn;
            }
        }
    }
}

// Row M5 second half for the odd (surface-curl) channels, by parts.  With the pooled grids
//   X0 = sum_e R~ (d_theta E_e) I_j,   X1 = -sum_e R~ ((1/sin) d_phi E_e) I_j       (edge_ring.cu / message.cu)
// the coupling  T_lm = int r.[grad E x grad I] Y_lm  (Eq.(57) PAPER.md:443 under Eq.(53)-(54)) equals, because the
// bracket of two functions integrates to zero over the sphere,
//   T_lm = -int I {E, Y_lm} = -int [ X1 d_theta Y_lm + X0 (1/sin) d_phi Y_lm ] dOmega ,
// and with (1/sin) d_phi Y_{l,+m} = -(m P~/sin) q_{-m}, (1/sin) d_phi Y_{l,-m} = +(m P~/sin) q_{+m}  (:679):
//   T_{l,+m} = sum_u w_u [ -dP~_l^m x1_{+m}(u) + (m P~_l^m/sin) x0_{-m}(u) ]
//   T_{l,-m} = sum_u w_u [ -dP~_l^m x1_{-m}(u) - (m P~_l^m/sin) x0_{+m}(u) ] .
// X0r, X1r: [M][J] shared azimuthal coefficients per grid row; WD, WS: [Uh][NTRI] weighted tables.
// Reflection x -> -x: m P~/sin has the parity (-1)^(l-m) of P~, d_theta P~ the opposite one.
template <int LB>
__device__ __forceinline__ void legendre_analysis_curl(const float* X0r, const float* X1r,
                                                       const float* __restrict__ WD, const float* __restrict__ WS,
                                                       float* __restrict__ out, int Lo2p, int NC, int lmax_out, int U,
                                                       int Uh, int NTRI, int J)
{
    constexpr int UHMAX = ((3 * LB + 2) / 2 + 1) / 2;
    // work item = (column, |m|, sign of m): T_{l,+m} needs x1_{+m} and x0_{-m}, T_{l,-m} needs x1_{-m} and x0_{+m}
    const int items = NC * (lmax_out + 1) * 2;
    for (int item = threadIdx.x; item < items; item += blockDim.x) {
        const int neg = item & 1;
        const int cm = item >> 1;
        const int col = cm / (lmax_out + 1);
        const int mm = cm - col * (lmax_out + 1);
        if (neg && mm == 0) continue;
        const int row1 = neg ? (LB + mm) : mm;  // row of X1 with the sign of the output m
        const int row0 = neg ? mm : (LB + mm);  // row of X0 with the opposite sign
        const float sgn0 = neg ? -1.f : 1.f;
        // [north + south, north - south][u']
        float f1[2][UHMAX], f0[2][UHMAX];
#pragma unroll
        for (int up = 0; up < UHMAX; ++up) {
            float n1 = 0.f, s1 = 0.f, n0 = 0.f, s0 = 0.f;
            if (up < Uh) {
                n1 = X1r[row1 * J + col * U + up];
                s1 = X1r[row1 * J + col * U + (U - 1 - up)];
                if (mm > 0) {
                    n0 = sgn0 * X0r[row0 * J + col * U + up];
                    s0 = sgn0 * X0r[row0 * J + col * U + (U - 1 - up)];
                }
            }
            f1[0][up] = n1 + s1;
            f1[1][up] = n1 - s1;
            f0[0][up] = n0 + s0;
            f0[1][up] = n0 - s0;
        }
        float* ocol = out + (size_t)col * Lo2p;
        // degrees in pairs so that the reflection parity of (l - m) is a compile-time constant:
        // par = 0: P~ symmetric, d_theta P~ antisymmetric under x -> -x; par = 1 the other way round
        for (int l0 = mm; l0 <= lmax_out; l0 += 2) {
#pragma unroll
            for (int par = 0; par < 2; ++par) {
                const int l = l0 + par;
                if (l > lmax_out) break;
                const int t0 = tri_index(l, mm);
                float acc = 0.f;
#pragma unroll
                for (int up = 0; up < UHMAX; ++up) {
                    if (up < Uh) {
                        const float wd = WD[up * NTRI + t0], ws = WS[up * NTRI + t0];
                        acc = fmaf(ws, f0[par][up], fmaf(-wd, f1[1 - par][up], acc));
                    }
                }
                ocol[l * l + l + (neg ? -mm : mm)] = acc;
            }
        }
    }
}

}  // namespace cgtp
