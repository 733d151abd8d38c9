// nbody_reg.cu -- nu-body on-site core for SMALL band limits with one thread per (atom, rank-channel) column
// and the whole chain of that column on registers, as onsite_reg.cu does for the bilinear product: for every
// Gauss-Legendre row u of the nu-body grid the Legendre synthesis of the nu factors (Eq.(36) :325), the forward real DFT
// of the nu coefficient vectors, the product of the nu grid values at the azimuth pair (v', V - v') and the inverse real
// DFT (Eq.(37)-(39) :327-:339), then the row's term of the quadrature (Eq.(40) :342) added to T.  Nothing is exchanged
// between threads: no barrier, no shared-memory round trip of the per-row coefficients (nbody.cu deals three stages over
// the 256 threads of a CTA with two barriers per tile).  A warp is a unit of its own: the nu H blocks of its 32 columns
// arrive by TMA bulk copies on the warp's mbarrier, T leaves through the warp's staging rows with a bulk store.
// Pairs for the packed FMAs: factors two at a time (the Legendre / Fourier table value is the broadcast scalar); an odd
// last factor and the inverse transform as (cosine row, sine row) pairs against the (qc, qs) table pair.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <mutex>

#include "onsite_reg.cuh"

namespace cgtp {

namespace {

struct NbRegPlan {
    int dev, lmax, lmax_out, nu;
    int floats, off_w, off_qi, off_wv, QP;
    const void* blob;  // device: P[U][NT4], WP[U][NT4], QI[Vh][QP] (qc, qs) pairs, WV[Vh]
};
std::mutex g_mu;
std::vector<NbRegPlan*> g_plans;

const NbRegPlan* get_plan_reg(const Plan* p)
{
    std::lock_guard<std::mutex> lk(g_mu);
    for (NbRegPlan* c : g_plans)
        if (c->dev == p->dev && c->lmax == p->lmax && c->lmax_out == p->lmax_out && c->nu == p->nu) return c;
    std::vector<float> tab;
    const int NT4 = reg_host_tables(p, false, tab);  // [P][WP] on the plan's nu-body grid
    const int QP = round_up(p->LB + 1, 2);
    NbRegPlan* c = new NbRegPlan;
    c->off_w = p->U * NT4;
    c->off_qi = (int)tab.size();
    tab.resize(tab.size() + (size_t)p->Vh * QP * 2, 0.f);
    for (int vp = 0; vp < p->Vh; ++vp)
        for (int m = 0; m <= p->LB; ++m) {
            tab[c->off_qi + ((size_t)vp * QP + m) * 2] = p->hQC[vp * p->QSTR + m];
            tab[c->off_qi + ((size_t)vp * QP + m) * 2 + 1] = p->hQS[vp * p->QSTR + m];
        }
    c->off_wv = (int)tab.size();
    tab.resize(tab.size() + round_up(p->Vh, 4), 0.f);
    for (int vp = 0; vp < p->Vh; ++vp) tab[c->off_wv + vp] = p->hWV[vp];
    void* d = nullptr;
    if (cudaMalloc(&d, tab.size() * 4) != cudaSuccess ||
        cudaMemcpy(d, tab.data(), tab.size() * 4, cudaMemcpyHostToDevice) != cudaSuccess) {
        set_error("nbody register core plan: device upload failed: %s", cudaGetErrorString(cudaGetLastError()));
        delete c;
        return nullptr;
    }
    c->dev = p->dev; c->lmax = p->lmax; c->lmax_out = p->lmax_out; c->nu = p->nu;
    c->floats = (int)tab.size();
    c->QP = QP;
    c->blob = d;
    g_plans.push_back(c);
    return c;
}

struct NbRegArgs {
    const float* tab;
    int tab_floats, off_w, off_qi, off_wv;
    const float* H;     // [nu][hfs]: rows of stride L2s, blocks padded to whole groups of 32 columns
    long long hfs;
    float* T;           // [groups * 32][Lo2s]
    long long ngroups;
    int U, Vh, L2, Lo2, L2s, Lo2s;
    int off_warp, warp_bytes, off_ts;
};

constexpr int kNbRegWarps = 4;

template <int LB, int NU>
__global__ void __launch_bounds__(32 * kNbRegWarps) nbody_reg_kernel(const NbRegArgs a)
{
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int NT = (LB + 1) * (LB + 2) / 2, NT4 = round_up(NT, 4), L2B = (LB + 1) * (LB + 1);
    constexpr int M = 2 * LB + 1, QP = round_up(LB + 1, 2);
    constexpr int NP = NU / 2, NR = NU % 2;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    pdl_launch_dependents();  // programmatic dependent launch, common.cuh
    float* tabs = reinterpret_cast<float*>(smem);
    for (int i = threadIdx.x; i < a.tab_floats; i += blockDim.x) tabs[i] = a.tab[i];  // the plan's tables: independent
    unsigned char* wr = smem + a.off_warp + (size_t)warp * a.warp_bytes;
    uint64_t* bar = reinterpret_cast<uint64_t*>(wr);
    float* hbuf = reinterpret_cast<float*>(wr + 16);
    float* Ts = reinterpret_cast<float*>(wr + a.off_ts);
    const int hfl = 32 * a.L2s;
    const uint32_t hbytes = (uint32_t)hfl * 4;
    if (lane == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncthreads();
    auto load_h = [&](long long g) {
        mbar_arrive_expect_tx(bar, NU * hbytes);
#pragma unroll
        for (int s = 0; s < NU; ++s) tma_load_span(hbuf + (size_t)s * hfl, a.H + (size_t)s * a.hfs + g * hfl, hbytes, bar);
    };
    const long long stride = (long long)gridDim.x * kNbRegWarps;
    long long g = (long long)blockIdx.x * kNbRegWarps + warp;
    pdl_wait();  // H is the predecessor's output
    if (lane == 0 && g < a.ngroups) load_h(g);
    const float* tabp = tabs;
    const float* tabw = tabs + a.off_w;
    const float4* QI = reinterpret_cast<const float4*>(tabs + a.off_qi);  // [Vh][QP] pairs (qc, qs): QP / 2 float4 per row
    const float* WV = tabs + a.off_wv;
    uint32_t phase = 0u;
    for (; g < a.ngroups; g += stride) {
        const long long gn = g + stride;
        mbar_wait(bar, phase);
        phase ^= 1u;
        const float* h = hbuf + lane * a.L2s;
        float T[L2B];
#pragma unroll
        for (int k = 0; k < L2B; ++k) T[k] = 0.f;

#pragma unroll 1
        for (int u = 0; u < a.U; ++u) {
            // ---- stage A: coefficient rows of grid row u for the NU factors
            float2 f2[NP > 0 ? NP : 1][M];  // (factor 2q, factor 2q+1)[row]
            float2 fr[LB + 1];              // odd last factor: (cosine row m, sine row m)
#pragma unroll
            for (int q = 0; q < NP; ++q)
#pragma unroll
                for (int r = 0; r < M; ++r) f2[q][r] = make_float2(0.f, 0.f);
#pragma unroll
            for (int m = 0; m <= LB; ++m) fr[m] = make_float2(0.f, 0.f);
#pragma unroll
            for (int j = 0; j < NT4; j += 4) {
                const float4 v0 = *reinterpret_cast<const float4*>(tabp + u * NT4 + j);
                const float t0[4] = {v0.x, v0.y, v0.z, v0.w};
#pragma unroll
                for (int hh = 0; hh < 4; ++hh) {
                    if (j + hh >= NT) break;
                    const int l = tri_l(j + hh), m = tri_m(j + hh);
                    const int ip = l * l + l + m, im = l * l + l - m;
                    const bool in = ip < a.L2;  // l <= lmax
                    const float2 p2 = make_float2(t0[hh], t0[hh]);
#pragma unroll
                    for (int q = 0; q < NP; ++q) {
                        const float* h0 = h + (size_t)(2 * q) * hfl;
                        const float* h1 = h0 + hfl;
                        const float2 xp = in ? make_float2(h0[ip], h1[ip]) : make_float2(0.f, 0.f);
                        f2[q][m] = ffma2(xp, p2, f2[q][m]);
                        if (m > 0) {
                            const float2 xm = in ? make_float2(h0[im], h1[im]) : make_float2(0.f, 0.f);
                            f2[q][LB + m] = ffma2(xm, p2, f2[q][LB + m]);
                        }
                    }
                    if (NR) {
                        const float* hl = h + (size_t)(NU - 1) * hfl;
                        const float2 x = in ? make_float2(hl[ip], m > 0 ? hl[im] : 0.f) : make_float2(0.f, 0.f);
                        fr[m] = ffma2(x, p2, fr[m]);
                    }
                }
            }
            // ---- stage B: forward DFT, product of the NU grid values at (v', V - v'), inverse DFT
            float2 t[LB + 1];  // (cosine row m, sine row m)
#pragma unroll
            for (int m = 0; m <= LB; ++m) t[m] = make_float2(0.f, 0.f);
#pragma unroll 1
            for (int vp = 0; vp < a.Vh; ++vp) {
                float2 qi[QP];
#pragma unroll
                for (int i = 0; i < QP / 2; ++i) {
                    const float4 v = QI[vp * (QP / 2) + i];
                    qi[2 * i] = make_float2(v.x, v.y);
                    qi[2 * i + 1] = make_float2(v.z, v.w);
                }
                float s1 = 1.f, s2 = 1.f;
#pragma unroll
                for (int q = 0; q < NP; ++q) {
                    float2 ce = make_float2(0.f, 0.f), so = make_float2(0.f, 0.f);
#pragma unroll
                    for (int m = 0; m <= LB; ++m) ce = ffma2(make_float2(qi[m].x, qi[m].x), f2[q][m], ce);
#pragma unroll
                    for (int m = 1; m <= LB; ++m) so = ffma2(make_float2(qi[m].y, qi[m].y), f2[q][LB + m], so);
                    s1 *= (ce.x + so.x) * (ce.y + so.y);  // grid point v'
                    s2 *= (ce.x - so.x) * (ce.y - so.y);  // mirrored grid point V - v'
                }
                if (NR) {
                    float2 cs = make_float2(0.f, 0.f);  // (cosine part, sine part)
#pragma unroll
                    for (int m = 0; m <= LB; ++m) cs = ffma2(qi[m], fr[m], cs);
                    s1 *= cs.x + cs.y;
                    s2 *= cs.x - cs.y;
                }
                const float w = WV[vp];
                const float2 spm = make_float2(w * (s1 + s2), w * (s1 - s2));
#pragma unroll
                for (int m = 0; m <= LB; ++m) t[m] = ffma2(qi[m], spm, t[m]);  // qs[0] = 0: t[0].y stays 0
            }
            // ---- stage C: this row's term of the quadrature
#pragma unroll
            for (int j = 0; j < NT4; j += 4) {
                const float4 v = *reinterpret_cast<const float4*>(tabw + u * NT4 + j);
                const float wv[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                for (int hh = 0; hh < 4; ++hh) {
                    if (j + hh >= NT) break;
                    const int l = tri_l(j + hh), m = tri_m(j + hh);
                    T[l * l + l + m] = fmaf(wv[hh], t[m].x, T[l * l + l + m]);
                    if (m > 0) T[l * l + l - m] = fmaf(wv[hh], t[m].y, T[l * l + l - m]);
                }
            }
        }

        __syncwarp();  // the rows of H are dead: refill the buffer while T is stored
        if (lane == 0) {
            if (gn < a.ngroups) load_h(gn);
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        }
        __syncwarp();
#pragma unroll
        for (int k = 0; k < L2B; ++k)
            if (k < a.Lo2) Ts[lane * a.Lo2s + k] = T[k];
        fence_async_smem();
        __syncwarp();
        if (lane == 0) {
            tma_store_1d(a.T + g * 32 * a.Lo2s, Ts, (uint32_t)(32 * a.Lo2s * 4));
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
    }
    if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

template <int LB, int NU>
int launch_t(const Plan* p, const NbRegPlan* c, const float* H, int64_t hfs, float* T, int64_t ncols, cudaStream_t st)
{
    NbRegArgs a;
    a.tab = reinterpret_cast<const float*>(c->blob);
    a.tab_floats = c->floats; a.off_w = c->off_w; a.off_qi = c->off_qi; a.off_wv = c->off_wv;
    a.H = H;
    a.hfs = hfs;
    a.T = T;
    a.ngroups = (ncols + 31) / 32;
    a.U = p->U; a.Vh = p->Vh; a.L2 = p->L2; a.Lo2 = p->Lo2; a.L2s = p->L2 | 1; a.Lo2s = p->Lo2 | 1;
    const int hbytes = NU * 32 * a.L2s * 4;
    a.off_ts = 16 + hbytes;
    a.warp_bytes = round_up(a.off_ts + 32 * a.Lo2s * 4, 128);
    a.off_warp = round_up(c->floats * 4, 128);
    const size_t smem = (size_t)a.off_warp + (size_t)kNbRegWarps * a.warp_bytes;
    auto kern = nbody_reg_kernel<LB, NU>;
    CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int ctas_per_sm = 0;
    CGTP_CUDA_CHECK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas_per_sm, kern, 32 * kNbRegWarps, smem));
    if (ctas_per_sm < 1) ctas_per_sm = 1;
    int64_t grid = (int64_t)num_sms() * ctas_per_sm;
    const int64_t need = (a.ngroups + kNbRegWarps - 1) / kNbRegWarps;
    if (grid > need) grid = need;
    LaunchScope scope(K_ONSITE_EVEN, st);
    CGTP_CUDA_CHECK(launch_pdl(kern, (unsigned)grid, 32u * kNbRegWarps, smem, st, a));
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

}  // namespace

// Measured (B200; core in us, this kernel against nbody_core_kernel): nu = 3 / 4 at lmax 3, N = C = 32, 16384 atoms: 84.5 /
// 127 vs 146 / 191; at lmax 6, N = C = 64, 4096 atoms: 199 / 437 vs 281 / 447.  (nu = 2 runs on the bilinear core.)
bool nbody_reg_supported(const Plan* p) { return p->LB <= 6 && p->nu >= 3 && p->nu <= 4; }

int launch_nbody_reg(const Plan* p, const float* H, int64_t hfs, float* T, int64_t ncols, cudaStream_t st)
{
    if (ncols <= 0) return CGTP_OK;
    const NbRegPlan* c = get_plan_reg(p);
    if (!c) return CGTP_ERR_CUDA;
    switch (p->LB * 8 + p->nu) {
#define CGTP_CASE(B)                                                           \
    case B * 8 + 3: return launch_t<B, 3>(p, c, H, hfs, T, ncols, st);         \
    case B * 8 + 4: return launch_t<B, 4>(p, c, H, hfs, T, ncols, st);
        CGTP_CASE(1) CGTP_CASE(2) CGTP_CASE(3) CGTP_CASE(4) CGTP_CASE(5) CGTP_CASE(6)
#undef CGTP_CASE
    }
    set_error("nbody register core: no kernel for band limit %d, body order %d", p->LB, p->nu);
    return CGTP_ERR_UNSUPPORTED;
}

}  // namespace cgtp
