// nbody.cu -- nu-body on-site core (end of Sec. VI): "The grid pointwise
// product extends to nu-body features through additional pointwise multiplications on the grid followed by a single
// inverse transform ... Higher-body-order products tighten this requirement linearly in the body order nu."
//
// Rows S2a, S2b, S3, S4a, S4b with nu factors instead of two, for NC (atom, rank-channel) columns per CTA:
// Legendre synthesis of every factor (Eq.(36) :325) -> per (column, grid row u): forward real DFT of the nu coefficient
// vectors (Eq.(37) :327), product of the nu grid values (Eq.(38) :332 with nu - 1 multiplications), inverse real DFT
// (Eq.(39) :339), all in registers -> Gauss-Legendre analysis (Eq.(40) :342).  The grid is the plan's
// U = ceil((nu lmax + lmax_out + 1)/2) x V = nu lmax + lmax_out + 1, on which the quadrature of the degree
// nu lmax + lmax_out integrand is exact.  Grid fields exist only in registers, the per-row azimuthal coefficients only
// in shared memory.  Pointwise (even) channels only: the curl pairing is bilinear (R23).
#include "sht.cuh"

namespace cgtp {

constexpr int kNbodyMaxBand = 20;
constexpr int kNbodyMaxNu = 4;

// H rows have the odd stride L2 | 1 (written so by S1): with lane = column the coefficient loads of the synthesis are
// then free of bank conflicts; a CTA's tile of every factor is one contiguous bulk copy of whole groups of 4 columns.
int nbody_hstride(const Plan* p) { return p->L2 | 1; }
// floats between the H blocks of consecutive factors (whole groups of 4 columns)
int64_t nbody_hfstride(const Plan* p, int64_t ncols) { return (ncols + 3) / 4 * 4 * (int64_t)nbody_hstride(p); }

bool nbody_supported(int LB, int nu) { return LB >= 1 && LB <= kNbodyMaxBand && nu >= 1 && nu <= kNbodyMaxNu; }

struct NbodySmem {
    // byte offsets into dynamic shared memory (all multiples of 16)
    int bar, tab, wp, qc, qs, qi, wv, hs, f, total;
    int tab_bytes, q_bytes, wv_bytes;
};

static NbodySmem nbody_smem_layout(const Plan* p, int NC)
{
    NbodySmem s;
    const int M = 2 * p->LB + 1;
    const int J = (NC * p->U) | 1;  // odd row stride: rows of different m fall into different banks
    s.tab_bytes = p->Uh * p->NTRI * 4;
    s.q_bytes = p->Vh * p->QSTR * 4;
    s.wv_bytes = round_up(p->Vh, 4) * 4;
    int off = 0;
    s.bar = off; off += 16;
    s.tab = off; off += s.tab_bytes;
    s.wp = off; off += s.tab_bytes;
    s.qc = off; off += s.q_bytes;
    s.qs = off; off += s.q_bytes;
    s.qi = off; off += p->Vh * round_up(p->LB + 1, 2) * 8;
    s.wv = off; off += s.wv_bytes;
    s.hs = off; off += p->nu * round_up(NC, 4) * nbody_hstride(p) * 4;
    s.f = off; off += round_up(p->nu * M * J, 4) * 4;
    s.total = off;
    return s;
}

// Row S2a for the NU factors (Eq.(36)).  Work item = (|m|, block of UB northern nodes, column), the column
// fastest: a warp shares |m| and the node block (the table loads are broadcasts, the loop trip counts agree), and items
// of the same cost sit next to one another, so that the strided item -> thread map deals every thread the same mix of
// cheap and expensive |m|.  Per degree: 2 NU coefficient loads and UB table loads feed 2 NU UB FMAs.  The sums are split
// into the parts even / odd under x -> -x (P~_l^m(-x) = (-1)^(l+m) P~_l^m(x)), one table row serves the node pair
// (u', U-1-u').  Table rows past Uh read by the last block are inside the shared-memory allocation; their sums are dropped.
template <int LB, int NU, int UB>
__device__ __forceinline__ void nbody_synthesis(const float* __restrict__ tab, const float* __restrict__ Hs,
                                                int h_in_stride, int L2p, float* F, int FS, int NC, int NCS, int lmax,
                                                int U, int Uh, int J)
{
    constexpr int NTRI = round_up((LB + 1) * (LB + 2) / 2, 4);
    const int nub = (Uh + UB - 1) / UB;
    const int items = (lmax + 1) * nub * NC;
    for (int item = threadIdx.x; item < items; item += blockDim.x) {
        const int mm = item / (nub * NC);
        const int rest = item - mm * (nub * NC);
        const int ub = rest / NC;
        const int col = rest - ub * NC;
        const float* hcol = Hs + (size_t)col * L2p;
        const float* trow = tab + (size_t)ub * UB * NTRI;
        float acc[NU][2][2][UB];  // [factor][+m, -m][parity of l - m][node]
#pragma unroll
        for (int a = 0; a < NU; ++a)
#pragma unroll
            for (int c = 0; c < 2; ++c)
#pragma unroll
                for (int d = 0; d < 2; ++d)
#pragma unroll
                    for (int e = 0; e < UB; ++e) acc[a][c][d][e] = 0.f;
        for (int l0 = mm; l0 <= lmax; l0 += 2) {
#pragma unroll
            for (int par = 0; par < 2; ++par) {
                const int l = l0 + par;
                if (l <= lmax) {
                    const int t = tri_index(l, mm);
                    const int c0 = l * l + l;
                    float pv[UB];
#pragma unroll
                    for (int e = 0; e < UB; ++e) pv[e] = trow[e * NTRI + t];
#pragma unroll
                    for (int a = 0; a < NU; ++a) {
                        const float hp = hcol[a * h_in_stride + c0 + mm];
                        const float hn = hcol[a * h_in_stride + c0 - mm];
#pragma unroll
                        for (int e = 0; e < UB; ++e) {
                            acc[a][0][par][e] = fmaf(pv[e], hp, acc[a][0][par][e]);
                            acc[a][1][par][e] = fmaf(pv[e], hn, acc[a][1][par][e]);
                        }
                    }
                }
            }
        }
#pragma unroll
        for (int e = 0; e < UB; ++e) {
            const int up = ub * UB + e;
            if (up < Uh) {
                const int jn = up * NCS + col, js = (U - 1 - up) * NCS + col;  // j = u * NCS + col: lanes = columns
#pragma unroll
                for (int a = 0; a < NU; ++a) {
                    float* Fa = F + (size_t)a * FS;
                    Fa[mm * J + jn] = acc[a][0][0][e] + acc[a][0][1][e];
                    Fa[mm * J + js] = acc[a][0][0][e] - acc[a][0][1][e];
                    if (mm > 0) {
                        Fa[(LB + mm) * J + jn] = acc[a][1][0][e] + acc[a][1][1][e];
                        Fa[(LB + mm) * J + js] = acc[a][1][0][e] - acc[a][1][1][e];
                    }
                }
            }
        }
    }
}

// Rows S2b + S3 + S4a for one (column, u): forward real DFT of the NU coefficient vectors, product of the NU grid
// values at the azimuth pair (v', V - v'), inverse real DFT.  F: NU fields [M][J] at distance FS; the result T[m]
// overwrites field 0 at [.][j].
// QI: interleaved Fourier table [Vh][QP] of pairs (qc[m], qs[m]), QP = LB + 1 rounded up to 2 pairs (16 bytes).
// Packed FP32 throughout (FFMA2): factors two at a time with the Fourier coefficient broadcast to both halves; an odd
// last factor and the inverse transform as (cosine part, sine part) pairs against the (qc, qs) pair.
template <int LB, int NU>
__device__ __forceinline__ void dft_nproduct_idft(float* F, int FS, int J, int j, const float2* __restrict__ QI,
                                                  const float* __restrict__ WV, int Vh)
{
    constexpr int M = 2 * LB + 1;
    constexpr int QP = round_up(LB + 1, 2);
    constexpr int NP = NU / 2, NR = NU % 2;
    float2 f2[NP > 0 ? NP : 1][M];  // (factor 2q, factor 2q+1)[row]
    float2 fr[LB + 1];              // odd last factor: (cosine row m, sine row m)
    float2 t[LB + 1];               // result: (cosine row m, sine row m)
#pragma unroll
    for (int q = 0; q < NP; ++q)
#pragma unroll
        for (int r = 0; r < M; ++r)
            f2[q][r] = make_float2(F[(size_t)(2 * q) * FS + r * J + j], F[(size_t)(2 * q + 1) * FS + r * J + j]);
    if (NR) {
        const float* Fl = F + (size_t)(NU - 1) * FS;
        fr[0] = make_float2(Fl[j], 0.f);
#pragma unroll
        for (int m = 1; m <= LB; ++m) fr[m] = make_float2(Fl[m * J + j], Fl[(LB + m) * J + j]);
    }
#pragma unroll
    for (int m = 0; m <= LB; ++m) t[m] = make_float2(0.f, 0.f);
    for (int vp = 0; vp < Vh; ++vp) {
        float2 qi[QP];
        const float4* src = reinterpret_cast<const float4*>(QI + vp * QP);
#pragma unroll
        for (int i = 0; i < QP / 2; ++i) {
            const float4 v = src[i];
            qi[2 * i] = make_float2(v.x, v.y);
            qi[2 * i + 1] = make_float2(v.z, v.w);
        }
        float s1 = 1.f, s2 = 1.f;
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            float2 ce = make_float2(0.f, 0.f), so = make_float2(0.f, 0.f);
#pragma unroll
            for (int m = 0; m <= LB; ++m) ce = __ffma2_rn(make_float2(qi[m].x, qi[m].x), f2[q][m], ce);
#pragma unroll
            for (int m = 1; m <= LB; ++m) so = __ffma2_rn(make_float2(qi[m].y, qi[m].y), f2[q][LB + m], so);
            s1 *= (ce.x + so.x) * (ce.y + so.y);  // grid point v'
            s2 *= (ce.x - so.x) * (ce.y - so.y);  // mirrored grid point V - v'
        }
        if (NR) {
            float2 cs = make_float2(0.f, 0.f);  // (cosine part, sine part)
#pragma unroll
            for (int m = 0; m <= LB; ++m) cs = __ffma2_rn(qi[m], fr[m], cs);
            s1 *= cs.x + cs.y;
            s2 *= cs.x - cs.y;
        }
        const float w = WV[vp];
        const float2 spm = make_float2(w * (s1 + s2), w * (s1 - s2));
#pragma unroll
        for (int m = 0; m <= LB; ++m) t[m] = __ffma2_rn(qi[m], spm, t[m]);  // qs[0] = 0: t[0].y stays 0
    }
    F[j] = t[0].x;
#pragma unroll
    for (int m = 1; m <= LB; ++m) {
        F[m * J + j] = t[m].x;
        F[(LB + m) * J + j] = t[m].y;
    }
}

// Row S4b (Eq.(40)): legendre_analysis of sht.cuh on the column-fastest row layout j = u * NCS + col.
// Work item = (column, |m|), |m| fastest: lanes read different coefficient rows (odd row stride J, no bank conflicts)
// and store neighbouring output coefficients.  North and south node are folded with the reflection parity (-1)^(l-m).
template <int LB, int UHMAX>
__device__ __forceinline__ void nbody_analysis(const float* Tr, const float* __restrict__ WP, float* __restrict__ out,
                                               int Lo2p, int NC, int NCS, int lmax_out, int U, int Uh, int J)
{
    constexpr int NTRI = round_up((LB + 1) * (LB + 2) / 2, 4);
    const int items = NC * (lmax_out + 1);
    for (int item = threadIdx.x; item < items; item += blockDim.x) {
        const int col = item / (lmax_out + 1);
        const int mm = item - col * (lmax_out + 1);
        float tp[2][UHMAX], tm[2][UHMAX];  // [+m, -m][u']: north + south, north - south
#pragma unroll
        for (int sg = 0; sg < 2; ++sg) {
            const int row = (sg == 0) ? mm : (LB + mm);
#pragma unroll
            for (int up = 0; up < UHMAX; ++up) {
                float n = 0.f, so = 0.f;
                if (up < Uh && !(sg == 1 && mm == 0)) {
                    n = Tr[row * J + up * NCS + col];
                    so = Tr[row * J + (U - 1 - up) * NCS + col];
                }
                tp[sg][up] = n + so;
                tm[sg][up] = n - so;
            }
        }
        float* ocol = out + (size_t)col * Lo2p;
        for (int l0 = mm; l0 <= lmax_out; l0 += 2) {
#pragma unroll
            for (int par = 0; par < 2; ++par) {
                const int l = l0 + par;
                if (l <= lmax_out) {
                    const int t = tri_index(l, mm);
                    float ap = 0.f, an = 0.f;
#pragma unroll
                    for (int up = 0; up < UHMAX; ++up) {
                        if (up < Uh) {
                            const float w = WP[up * NTRI + t];
                            ap = fmaf(w, par ? tm[0][up] : tp[0][up], ap);
                            an = fmaf(w, par ? tm[1][up] : tp[1][up], an);
                        }
                    }
                    ocol[l * l + l + mm] = ap;
                    if (mm > 0) ocol[l * l + l - mm] = an;
                }
            }
        }
    }
}

template <int LB, int NU>
__global__ void __launch_bounds__(256, (LB <= 8 ? 2 : 1)) nbody_core_kernel(Plan p, NbodySmem lay, const float* __restrict__ H,
                                                            long long hfs, float* __restrict__ T, long long ncols, int NC)
{
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int M = 2 * LB + 1;
    constexpr int UHMAX = (((NU + 1) * LB + 2) / 2 + 1) / 2;  // Uh for lmax = lmax_out = LB
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + lay.bar);
    float* tab = reinterpret_cast<float*>(smem + lay.tab);
    float* wp = reinterpret_cast<float*>(smem + lay.wp);
    float* qc = reinterpret_cast<float*>(smem + lay.qc);
    float* qs = reinterpret_cast<float*>(smem + lay.qs);
    float* wv = reinterpret_cast<float*>(smem + lay.wv);
    float* hs = reinterpret_cast<float*>(smem + lay.hs);
    float* F = reinterpret_cast<float*>(smem + lay.f);

    const long long col0 = (long long)blockIdx.x * NC;
    const int nc = (int)((ncols - col0 < NC) ? (ncols - col0) : NC);
    const int J = (NC * p.U) | 1;
    const int FS = M * J;
    const int hstr = p.L2 | 1;
    const int NC4 = round_up(NC, 4);
    const int hbytes = round_up(nc, 4) * hstr * 4;  // whole groups of 4 columns (16-byte granularity); H is padded

    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const uint32_t total = 2 * lay.tab_bytes + 2 * lay.q_bytes + lay.wv_bytes + NU * hbytes;
        mbar_arrive_expect_tx(bar, total);
        tma_load_span(tab, p.PT, lay.tab_bytes, bar);
        tma_load_span(wp, p.WP, lay.tab_bytes, bar);
        tma_load_span(qc, p.QC, lay.q_bytes, bar);
        tma_load_span(qs, p.QS, lay.q_bytes, bar);
        tma_load_span(wv, p.WV, lay.wv_bytes, bar);
#pragma unroll
        for (int s = 0; s < NU; ++s)
            tma_load_span(hs + (size_t)s * NC4 * hstr, H + (size_t)s * hfs + (size_t)col0 * hstr, hbytes, bar);
    }
#pragma unroll
    for (int s = 0; s < NU; ++s) zero_high_rows<LB>(F + (size_t)s * FS, p.lmax, J);
    mbar_wait(bar, 0);
    // interleaved Fourier table for the packed azimuthal stage (read after the barrier that ends the synthesis)
    float2* qi = reinterpret_cast<float2*>(smem + lay.qi);
    {
        constexpr int QP = round_up(LB + 1, 2);
        for (int i = threadIdx.x; i < p.Vh * QP; i += blockDim.x) {
            const int vp = i / QP, m = i - vp * QP;
            qi[i] = (m <= LB) ? make_float2(qc[vp * p.QSTR + m], qs[vp * p.QSTR + m]) : make_float2(0.f, 0.f);
        }
    }

    // ---- S2a: Legendre synthesis of the NU factors
    nbody_synthesis<LB, NU, 4>(tab, hs, NC4 * hstr, hstr, F, FS, nc, NC, p.lmax, p.U, p.Uh, J);
    __syncthreads();

    // ---- S2b + S3 + S4a: one (column, u) per thread
    const int rows = nc * p.U;
    for (int item = threadIdx.x; item < rows; item += blockDim.x) {
        const int u = item / nc, col = item - u * nc;
        dft_nproduct_idft<LB, NU>(F, FS, J, u * NC + col, qi, wv, p.Vh);
    }
    __syncthreads();

    // ---- S4b: Gauss-Legendre analysis
    nbody_analysis<LB, UHMAX>(F, wp, T + col0 * p.Lo2p, p.Lo2p, nc, NC, p.lmax_out, p.U, p.Uh, J);
}

template <int LB, int NU>
static int launch_nbody_t(const Plan* p, const float* H, float* T, int64_t ncols, cudaStream_t st)
{
    const int M = 2 * p->LB + 1;
    // columns per CTA: fill ~112 KB of shared memory (two CTAs per SM), at least 1 column
    NbodySmem fixed = nbody_smem_layout(p, 4);  // includes the padding of the H tiles to whole groups of 4 columns
    const int percol = NU * nbody_hstride(p) * 4 + NU * M * p->U * 4;
    int NC = (112 * 1024 - fixed.total - 64) / percol;
    if (NC < 4) NC = (220 * 1024 - fixed.total - 64) / percol;
    if (NC < 1) { set_error("nbody core: shared memory too small for lmax=%d nu=%d", p->lmax, NU); return CGTP_ERR_UNSUPPORTED; }
    if (NC > 128) NC = 128;
    // at least ~2 CTAs per SM when the problem is small
    while (NC > 8 && (ncols + NC - 1) / NC < 296) NC /= 2;
    if ((int64_t)NC > ncols) NC = (int)ncols;
    {
        // every stage deals its items over the 256 threads in strided passes: among the column counts near the one
        // that fills shared memory take the one with the fewest idle thread slots in the last passes (estimated
        // instruction cost per item: synthesis ~ 10 NU per degree, transform ~ Vh (2 NU + 2) LB, analysis ~ 3 Uh per degree)
        const int nub = (p->Uh + 3) / 4;
        const double c_syn = 10.0 * NU * (p->lmax + 2) / 2.0, c_dft = (double)p->Vh * (2 * NU + 2) * (p->LB + 1),
                     c_ana = 3.0 * p->Uh * (p->lmax_out + 2) / 2.0;
        auto passes = [](int items) { return (items + 255) / 256; };
        int best = NC;
        double bestc = 1e300;
        for (int n = NC; n >= 1 && n >= NC * 2 / 3; --n) {
            const double c = (passes((p->lmax + 1) * nub * n) * c_syn + passes(n * p->U) * c_dft +
                              passes(n * (p->lmax_out + 1)) * c_ana) / n;
            if ((n % 4 == 0 || n < 4) && c < bestc * 0.999) { bestc = c; best = n; }
        }
        NC = best;
    }
    if (NC >= 4 && (int64_t)NC < ncols) NC &= ~3;  // tiles start at 16-byte boundaries of H
    if (NC < 4 && (int64_t)NC < ncols) { set_error("nbody core: fewer than 4 columns per CTA fit shared memory (lmax=%d nu=%d)", p->lmax, NU); return CGTP_ERR_UNSUPPORTED; }
    NbodySmem lay = nbody_smem_layout(p, NC);
    auto kern = nbody_core_kernel<LB, NU>;
    CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, lay.total));
    int64_t grid = (ncols + NC - 1) / NC;
    LaunchScope scope(K_ONSITE_EVEN, st);
    kern<<<(unsigned)grid, 256, lay.total, st>>>(*p, lay, H, (long long)nbody_hfstride(p, ncols), T, (long long)ncols, NC);
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

#define CGTP_FOR_EACH_NBODY_BAND(X) X(1) X(2) X(3) X(4) X(5) X(6) X(8) X(10) X(12) X(16) X(20)

int launch_nbody(const Plan* p, const float* H, float* T, int64_t ncols, cudaStream_t st)
{
    if (ncols <= 0) return CGTP_OK;
    if (!nbody_supported(p->LB, p->nu)) {
        set_error("nbody core: band limit %d / body order %d not supported (max %d / %d)", p->LB, p->nu, kNbodyMaxBand,
                  kNbodyMaxNu);
        return CGTP_ERR_UNSUPPORTED;
    }
    switch (p->LB * 8 + p->nu) {
#define CGTP_CASE(B)                                                        \
    case B * 8 + 1: return launch_nbody_t<B, 1>(p, H, T, ncols, st);        \
    case B * 8 + 2: return launch_nbody_t<B, 2>(p, H, T, ncols, st);        \
    case B * 8 + 3: return launch_nbody_t<B, 3>(p, H, T, ncols, st);        \
    case B * 8 + 4: return launch_nbody_t<B, 4>(p, H, T, ncols, st);
        CGTP_FOR_EACH_NBODY_BAND(CGTP_CASE)
#undef CGTP_CASE
    }
    set_error("nbody core: no kernel for band limit %d, body order %d", p->LB, p->nu);
    return CGTP_ERR_UNSUPPORTED;
}

}  // namespace cgtp
