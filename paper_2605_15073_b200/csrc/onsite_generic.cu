// onsite.cu -- fused on-site core (rows S2a, S2b, S3, S4a, S4b of SURVEY.md 8(a)):
// Legendre synthesis -> phi synthesis -> pointwise product (even channels, Eq.(38)) or
// surface-curl pairing (odd channels, Eq.(11) :107 in theta-form) -> inverse phi transform ->
// Gauss-Legendre analysis, for NC (atom, rank-channel) columns per CTA.  The grid fields exist only
// in registers, the per-row azimuthal coefficients only in shared memory: nothing of size U*V ever
// goes to HBM (the paper's own implementation round-trips it after every stage).
//
// Odd channels are evaluated as two product terms that share the inverse transform by linearity:
//   {A,B} = A_theta * B_phi - A_phi * B_theta,  A_theta = d_theta A,  A_phi = (1/sin theta) d_phi A.
#include "sht.cuh"

namespace cgtp {

struct OnsiteSmem {
    // byte offsets into dynamic shared memory (all multiples of 16)
    int bar, tab0, tab1, wp, qc, qs, wv, hs, f, total;
    int tab_bytes, q_bytes, wv_bytes;
};

static OnsiteSmem onsite_smem_layout(const Plan* p, bool odd, int NC)
{
    OnsiteSmem s;
    const int M = 2 * p->LB + 1;
    const int J = (NC * p->U) | 1;  // odd row stride: rows of different m fall into different banks
    const int nterm = odd ? 2 : 1;
    s.tab_bytes = p->Uh * p->NTRI * 4;
    s.q_bytes = p->Vh * p->QSTR * 4;
    s.wv_bytes = round_up(p->Vh, 4) * 4;
    int off = 0;
    s.bar = off; off += 16;
    s.tab0 = off; off += s.tab_bytes;
    s.tab1 = off; off += odd ? s.tab_bytes : 0;
    s.wp = off; off += s.tab_bytes;
    s.qc = off; off += s.q_bytes;
    s.qs = off; off += s.q_bytes;
    s.wv = off; off += s.wv_bytes;
    s.hs = off; off += 2 * NC * p->L2p * 4;
    s.f = off; off += round_up(nterm * 2 * M * J, 4) * 4;
    s.total = off;
    return s;
}

template <int LB, bool ODD>
__global__ void __launch_bounds__(256) onsite_core_kernel(Plan p, OnsiteSmem lay, const float* __restrict__ Ha,
                                                         const float* __restrict__ Hb, float* __restrict__ T,
                                                         long long ncols, int NC)
{
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int M = 2 * LB + 1;
    constexpr int NTERM = ODD ? 2 : 1;
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + lay.bar);
    float* tab0 = reinterpret_cast<float*>(smem + lay.tab0);
    float* tab1 = reinterpret_cast<float*>(smem + lay.tab1);
    float* wp = reinterpret_cast<float*>(smem + lay.wp);
    float* qc = reinterpret_cast<float*>(smem + lay.qc);
    float* qs = reinterpret_cast<float*>(smem + lay.qs);
    float* wv = reinterpret_cast<float*>(smem + lay.wv);
    float* hs = reinterpret_cast<float*>(smem + lay.hs);
    float* F = reinterpret_cast<float*>(smem + lay.f);

    const long long col0 = (long long)blockIdx.x * NC;
    const int nc = (int)((ncols - col0 < NC) ? (ncols - col0) : NC);
    const int J = (NC * p.U) | 1;  // odd row stride (matches the host layout)
    const int hbytes = nc * p.L2p * 4;

    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const uint32_t total = (ODD ? 3 : 2) * lay.tab_bytes + 2 * lay.q_bytes + lay.wv_bytes + 2 * hbytes;
        mbar_arrive_expect_tx(bar, total);
        tma_load_span(tab0, ODD ? p.DT : p.PT, lay.tab_bytes, bar);
        if (ODD) tma_load_span(tab1, p.ST, lay.tab_bytes, bar);
        tma_load_span(wp, p.WP, lay.tab_bytes, bar);
        tma_load_span(qc, p.QC, lay.q_bytes, bar);
        tma_load_span(qs, p.QS, lay.q_bytes, bar);
        tma_load_span(wv, p.WV, lay.wv_bytes, bar);
        tma_load_span(hs, Ha + col0 * p.L2p, hbytes, bar);
        tma_load_span(hs + NC * p.L2p, Hb + col0 * p.L2p, hbytes, bar);
    }
    // F(term, which) : [M][J]
    auto Fp = [&](int term, int which) { return F + (size_t)(term * 2 + which) * M * J; };
#pragma unroll
    for (int i = 0; i < NTERM * 2; ++i) zero_high_rows<LB>(F + (size_t)i * M * J, p.lmax, J);
    mbar_wait(bar, 0);

    // ---- S2a: Legendre synthesis of both factors
    if (!ODD) {
        const LegDst dst[2][2] = {{{Fp(0, 0), 1.f}, {nullptr, 0.f}}, {{Fp(0, 1), 1.f}, {nullptr, 0.f}}};
        legendre_synthesis<LB, false, 2, (LB <= 8 ? 4 : 2)>(tab0, nullptr, hs, NC * p.L2p, p.L2p, dst, nc, p.lmax, p.U,
                                                            p.Uh, p.NTRI, J);
    } else {
        // term 0: (A_theta, B_phi); term 1: (-A_phi, B_theta)
        const LegDst dst[2][2] = {{{Fp(0, 0), 1.f}, {Fp(1, 0), -1.f}}, {{Fp(1, 1), 1.f}, {Fp(0, 1), 1.f}}};
        legendre_synthesis<LB, true, 2, 2>(tab0, tab1, hs, NC * p.L2p, p.L2p, dst, nc, p.lmax, p.U, p.Uh, p.NTRI, J);
    }
    __syncthreads();

    // ---- S2b + S3 + S4a: one (term, column, u) per thread
    const int rows = nc * p.U;
    for (int item = threadIdx.x; item < NTERM * rows; item += blockDim.x) {
        const int term = item / rows;
        const int j = item - term * rows;
        dft_product_idft<LB>(Fp(term, 0), Fp(term, 1), J, j, qc, qs, wv, p.Vh);
    }
    __syncthreads();

    // ---- S4b: Gauss-Legendre analysis
    legendre_analysis<LB>(Fp(0, 0), ODD ? Fp(1, 0) : nullptr, wp, T + col0 * p.Lo2p, p.Lo2p, nc, p.lmax_out, p.U, p.Uh,
                          p.NTRI, J);
}

template <int LB, bool ODD>
static int launch_onsite_t(const Plan* p, const float* Ha, const float* Hb, float* T, int64_t ncols, cudaStream_t st)
{
    const bool odd = ODD;
    const int M = 2 * p->LB + 1;
    const int nterm = odd ? 2 : 1;
    // columns per CTA: fill ~100 KB of shared memory (two CTAs per SM), at least 1 column
    OnsiteSmem fixed = onsite_smem_layout(p, odd, 0);
    const int percol = 2 * p->L2p * 4 + nterm * 2 * M * p->U * 4;
    int budget = 100 * 1024;
    int NC = (budget - fixed.total - 64) / percol;
    if (NC < 4) {
        budget = 220 * 1024;
        NC = (budget - fixed.total - 64) / percol;
    }
    if (NC < 1) { set_error("onsite core: shared memory too small for lmax=%d", p->lmax); return CGTP_ERR_UNSUPPORTED; }
    if (NC > 128) NC = 128;
    if ((int64_t)NC > ncols) NC = (int)ncols;
    OnsiteSmem lay = onsite_smem_layout(p, odd, NC);
    auto kern = onsite_core_kernel<LB, ODD>;
    CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, lay.total));
    int64_t grid = (ncols + NC - 1) / NC;
    LaunchScope scope(odd ? K_ONSITE_ODD : K_ONSITE_EVEN, st);
    kern<<<(unsigned)grid, 256, lay.total, st>>>(*p, lay, Ha, Hb, T, (long long)ncols, NC);
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

int launch_onsite_generic(const Plan* p, bool odd, const float* Ha, const float* Hb, float* T, int64_t ncols,
                       cudaStream_t st)
{
    if (ncols <= 0) return CGTP_OK;
    switch (p->LB) {
#define CGTP_CASE(B)                                                                   \
    case B:                                                                            \
        return odd ? launch_onsite_t<B, true>(p, Ha, Hb, T, ncols, st)                 \
                   : launch_onsite_t<B, false>(p, Ha, Hb, T, ncols, st);
        CGTP_FOR_EACH_BAND(CGTP_CASE)
#undef CGTP_CASE
    }
    set_error("onsite core: no kernel for band limit %d", p->LB);
    return CGTP_ERR_UNSUPPORTED;
}

}  // namespace cgtp
