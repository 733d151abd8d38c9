// sht_fast.cu -- lane = column form of node synthesis (row M2 of SURVEY.md 8(a); Eq.(49), (51) PAPER.md:404-:410) for
// band limits whose 32-column tile fits shared memory.  Same mathematics and the same folding as the generic kernel of
// message.cu / sht.cuh; what differs is the mapping:
//   * a CTA works on groups of 32 (node, rank-channel) columns, lane = column: every shared-memory array has the
//     column as its fastest index or an odd column stride, so no access has a bank conflict, and every table value is
//     a warp-wide broadcast (one 128-bit load feeds four packed FMAs);
//   * packed FP32 FMAs: the pair is (+m, -m) in the Legendre stage and (north row u, south row U-1-u) in the
//     Fourier stage;
//   * the grid tile of the group is staged in shared memory and written to HBM with coalesced stores.
// The generic kernel shares one table row among lanes of different m (conflicts, divergent trip counts) and runs the
// shared-memory pipe at 78 % for 25 % FMA-pipe activity (profiles/r01f_message_config4_ncu.txt); this one is
// issue-bound at 61 % (profiles/r01g_message_config4_ncu.txt).  The per-receiver analysis (M5) still uses the generic form.
#include <algorithm>

#include "sht.cuh"

namespace cgtp {

constexpr int SF_THREADS = 256;
constexpr int SF_WARPS = SF_THREADS / 32;

struct SfLayout {
    int ptt, qc, qs, hs, f, gt, total;  // float offsets
    int UP, GS, HS;
};

__host__ __device__ inline int sf_warp_of_item(int m)
{
    // items of decreasing cost dealt boustrophedon over the warps
    const int r = m / SF_WARPS, k = m % SF_WARPS;
    return (r & 1) ? SF_WARPS - 1 - k : k;
}

static SfLayout sf_layout(const Plan* p, int hstride, int nfield)
{
    SfLayout s;
    const int M = 2 * p->LB + 1;
    const int ntri = (p->LB + 1) * (p->LB + 2) / 2;
    s.UP = round_up(((3 * p->LB + 2) / 2 + 1) / 2, 4);  // compile-time bound of the kernels (Uh <= UHMAX(LB))
    s.GS = p->UVp | 1;
    s.HS = hstride;
    int off = 0;
    s.ptt = off; off += round_up(nfield * ntri * s.UP, 4);
    s.qc = s.qs = off;  // the azimuthal tables are a kernel parameter (QParam)
    s.f = off; off += nfield * M * p->U * 32;
    s.gt = off; off += std::max(round_up(32 * s.GS, 4), round_up(32 * hstride, 4));
    s.hs = s.gt;  // the coefficients are dead once the Legendre stage has run; the grid tile reuses their space
    s.total = off;
    return s;
}

// ------------------------------------------------------------------------------------------------
// M2: value grid field of 32 columns per group.  H: [col][hstride] (hstride odd), G: [col][UVp].
// ------------------------------------------------------------------------------------------------
template <int LB>
__global__ void __launch_bounds__(SF_THREADS) synth_fast_kernel(Plan p, SfLayout lay, const __grid_constant__ QParam<LB> qp,
                                                               const float* __restrict__ H, float* __restrict__ G,
                                                               long long ncols)
{
    extern __shared__ __align__(16) float sm[];
    constexpr int M = 2 * LB + 1;
    constexpr int QSTR = round_up(LB + 1, 4);
    constexpr int UHMAX = ((3 * LB + 2) / 2 + 1) / 2;
    constexpr int UP = round_up(UHMAX, 4);
    float* PTt = sm + lay.ptt;  // [tri][UP]
    float* Hs = sm + lay.hs;    // [32][HS]
    float* F = sm + lay.f;      // [M][U][32]
    float* Gt = sm + lay.gt;    // [32][GS]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int U = p.U, Uh = p.Uh, V = p.V, Vh = p.Vh, UVp = p.UVp, lmax = p.lmax;
    const int HS = lay.HS, GS = lay.GS;
    constexpr int ntri = (LB + 1) * (LB + 2) / 2;

    pdl_launch_dependents();  // programmatic dependent launch, common.cuh: the table set-up below touches only the plan
    for (int i = tid; i < ntri * UP; i += SF_THREADS) {
        const int t = i / UP, u = i - t * UP;
        PTt[i] = (u < Uh) ? p.PT[u * p.NTRI + t] : 0.f;
    }
    // coefficient rows above lmax (kernel band limit LB > lmax) stay zero for the whole kernel
    for (int i = tid; i < M * U * 32; i += SF_THREADS) F[i] = 0.f;

    pdl_wait();  // H is the predecessor's output, G may still be read by an earlier kernel of the stream
    const long long ngroups = (ncols + 31) / 32;
    for (long long g = blockIdx.x; g < ngroups; g += gridDim.x) {
        __syncthreads();
        {
            const float* src = H + g * 32 * HS;  // the buffer is padded to whole groups
            for (int i = tid; i < 32 * HS; i += SF_THREADS) Hs[i] = src[i];
        }
        __syncthreads();

        // ---- Legendre synthesis: warp item = |m|, lane = column, pair = (+m, -m)
        for (int m = 0; m <= lmax; ++m) {
            if (sf_warp_of_item(m) != warp) continue;
            const float* h = Hs + lane * HS;
            float2 acc[2][UP];
#pragma unroll
            for (int e = 0; e < UP; ++e) acc[0][e] = acc[1][e] = make_float2(0.f, 0.f);
            for (int l = m; l <= lmax; l += 2) {
#pragma unroll
                for (int par = 0; par < 2; ++par) {
                    const int ll = l + par;
                    if (ll > lmax) break;
                    const float4* tab = reinterpret_cast<const float4*>(PTt + tri_index(ll, m) * UP);
                    const float2 x = make_float2(h[ll * ll + ll + m], h[ll * ll + ll - m]);
#pragma unroll
                    for (int e = 0; e < UP; e += 4) {
                        const float4 t4 = tab[e / 4];
                        acc[par][e] = __ffma2_rn(x, make_float2(t4.x, t4.x), acc[par][e]);
                        acc[par][e + 1] = __ffma2_rn(x, make_float2(t4.y, t4.y), acc[par][e + 1]);
                        acc[par][e + 2] = __ffma2_rn(x, make_float2(t4.z, t4.z), acc[par][e + 2]);
                        acc[par][e + 3] = __ffma2_rn(x, make_float2(t4.w, t4.w), acc[par][e + 3]);
                    }
                }
            }
            // P~(-x) = (-1)^(l+m) P~(x): north = even + odd part, south = even - odd part
#pragma unroll
            for (int e = 0; e < UP; ++e) {
                if (e < Uh) {
                    const float2 n = __fadd2_rn(acc[0][e], acc[1][e]);
                    const float2 s = __fadd2_rn(acc[0][e], make_float2(-acc[1][e].x, -acc[1][e].y));
                    F[(m * U + e) * 32 + lane] = n.x;
                    F[(m * U + (U - 1 - e)) * 32 + lane] = s.x;
                    if (m > 0) {
                        F[((LB + m) * U + e) * 32 + lane] = n.y;
                        F[((LB + m) * U + (U - 1 - e)) * 32 + lane] = s.y;
                    }
                }
            }
        }
        __syncthreads();
        // padding of every grid field is written as zeros (the edge kernel streams whole float4s)
        for (int i = tid; i < 32 * (GS - p.UV); i += SF_THREADS) {
            const int c = i / (GS - p.UV), k = i - c * (GS - p.UV);
            Gt[c * GS + p.UV + k] = 0.f;
        }

        // ---- azimuthal synthesis: warp item = row pair (u, U-1-u), lane = column, pair = (north, south)
        for (int e = warp; e < Uh; e += SF_WARPS) {
            const int un = e, us = U - 1 - e;
            float2 f[M];
#pragma unroll
            for (int r = 0; r < M; ++r) f[r] = make_float2(F[(r * U + un) * 32 + lane], F[(r * U + us) * 32 + lane]);
            float* gn = Gt + lane * GS + un * V;
            float* gs = Gt + lane * GS + us * V;
            // two azimuths per pass: four independent accumulation chains.  The azimuth loop is fully unrolled over the
            // largest table of the band limit, so every table value is a constant-bank operand (QParam, sht.cuh): no
            // shared-memory wavefronts for the tables (this stage ran the shared-memory pipe above the FMA pipe)
#pragma unroll
            for (int vp0 = 0; vp0 < QParam<LB>::VHMAX; vp0 += 2) {
                if (vp0 >= Vh) break;
                float2 ce[2], so[2];
#pragma unroll
                for (int w = 0; w < 2; ++w) ce[w] = so[w] = make_float2(0.f, 0.f);
                const bool two = vp0 + 1 < Vh;
#pragma unroll
                for (int m = 0; m <= LB; ++m) {
#pragma unroll
                    for (int w = 0; w < 2; ++w) {
                        if (vp0 + w >= QParam<LB>::VHMAX) continue;
                        const float c = qp.qc[(vp0 + w) * QSTR + m];
                        ce[w] = __ffma2_rn(f[m], make_float2(c, c), ce[w]);
                        if (m >= 1) {
                            const float sn = qp.qs[(vp0 + w) * QSTR + m];
                            so[w] = __ffma2_rn(f[LB + m], make_float2(sn, sn), so[w]);
                        }
                    }
                }
#pragma unroll
                for (int w = 0; w < 2; ++w) {
                    if (w && !two) break;
                    const int vp = vp0 + w;
                    const float2 a = __fadd2_rn(ce[w], so[w]), b = __fadd2_rn(ce[w], make_float2(-so[w].x, -so[w].y));
                    gn[vp] = a.x;
                    gs[vp] = a.y;
                    if (vp > 0) {  // mirrored azimuth V - v' (a self-mirrored v' writes the same value twice: so = 0)
                        gn[V - vp] = b.x;
                        gs[V - vp] = b.y;
                    }
                }
            }
        }
        __syncthreads();

        // ---- coalesced store of the group's grid fields
        const long long col0 = g * 32;
        const int nc = (int)((ncols - col0 < 32) ? (ncols - col0) : 32);
        float* dst = G + col0 * UVp;
        for (int c = warp; c < nc; c += SF_WARPS)
            for (int k = lane; k < UVp; k += 32) dst[(size_t)c * UVp + k] = Gt[c * GS + k];
    }
}

bool synth_fast_supported(const Plan* p)
{
    const SfLayout lay = sf_layout(p, p->L2 | 1, 1);
    // measured against the generic kernel (4096 nodes x 128 channels): 0.71x / 0.90x / 0.85x / 0.89x of its time at band
    // limits 5 / 6 / 8 / 10; slower at <= 4 (too little work per 32-column group) and at 12 (one CTA per SM)
    return p->LB >= 5 && p->LB <= 10 && (size_t)lay.total * 4 <= 150 * 1024;
}

template <int LB>
static int launch_synth_fast_t(const Plan* p, Kind kind, const float* H, int hstride, float* G, int64_t ncols, cudaStream_t st)
{
    const SfLayout lay = sf_layout(p, hstride, 1);
    const size_t smem = (size_t)lay.total * 4;
    auto kern = synth_fast_kernel<LB>;
    CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = (int)((220 * 1024) / (smem + 1024));
    if (per_sm < 1) per_sm = 1;
    if (per_sm > 4) per_sm = 4;
    const int64_t ngroups = (ncols + 31) / 32;
    const int grid = (int)std::min<int64_t>(ngroups, (int64_t)148 * per_sm);
    LaunchScope scope(kind, st);
    QParam<LB> qp;
    fill_qparam<LB>(p, qp);
    CGTP_CUDA_CHECK(launch_pdl(kern, (unsigned)grid, (unsigned)SF_THREADS, smem, st, *p, lay, qp, H, G, (long long)ncols));
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

int launch_node_synth_fast(const Plan* p, bool odd, const float* H, int hstride, float* G, int64_t ncols, cudaStream_t st)
{
    if (ncols <= 0) return CGTP_OK;
    const Kind kind = odd ? K_NODE_SYNTH_ODD : K_NODE_SYNTH_EVEN;
    switch (p->LB) {
#define CGTP_CASE(B) \
    case B:          \
        return launch_synth_fast_t<B>(p, kind, H, hstride, G, ncols, st);
        CGTP_CASE(5) CGTP_CASE(6) CGTP_CASE(8) CGTP_CASE(10)
#undef CGTP_CASE
    }
    set_error("fast node synthesis: no kernel for band limit %d", p->LB);
    return CGTP_ERR_UNSUPPORTED;
}

}  // namespace cgtp
