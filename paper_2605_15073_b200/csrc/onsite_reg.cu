// onsite_reg.cu -- on-site core (rows S2a, S2b, S3, S4a, S4b of SURVEY.md 8(a)) for SMALL band limits with one thread per
// (atom, rank-channel) column and the whole transform chain of that column in registers:
//   for every Gauss-Legendre row u:   Legendre synthesis of the row (Eq.(36))
//                                  -> azimuthal synthesis, product (Eq.(38) :332) or surface-curl pairing (Eq.(11) :107),
//                                     inverse azimuthal transform (Eq.(37), (39) :327, :339; stage_b_regs)
//                                  -> the row's term of the Gauss-Legendre quadrature (Eq.(40) :342) added to T.
// Against onsite_fast_kernel (warps split each stage by a static schedule, the grid rows of a group travel through shared
// memory, three CTA-wide barriers per group) nothing is exchanged between threads: no barrier, no shared-memory round trip of
// the Fourier-Legendre coefficients, no ragged per-m schedule.  At small band limits those, not the arithmetic, were the
// cost (lmax 4, configs[3]: 7 grid rows on 4-8 warps).  The price is the x -> -x folding of the Legendre stages (a row
// needs all (l, m) terms: 2 x the FMAs of stages A and C, which are a small part at these sizes) and registers: the
// coefficient vectors H (LB <= 4) and T of a column live in registers, so the form stops at band limit 6.
//
// A warp is a unit of its own: its 32 columns' H block arrives by TMA bulk copy on the warp's mbarrier, T leaves through
// the warp's staging rows with a TMA bulk store; Legendre table rows are warp-uniform broadcast loads, the azimuthal tables
// are constant-bank operands (CoreQParam).
#include <algorithm>
#include <cmath>
#include <cstring>
#include <mutex>

#include "onsite_reg.cuh"

namespace cgtp {

int reg_host_tables(const Plan* p, bool odd, std::vector<float>& tab)
{
    const int LB = p->LB, U = p->U, LL = LB + 1;
    const int NT = (LB + 1) * (LB + 2) / 2, NT4 = round_up(NT, 4);
    std::vector<double> x, w, P;
    gauss_legendre(U, x, w);
    legendre_values(U, LB, x, P);
    auto at = [&](int u, int l, int m) -> double { return P[((size_t)u * LL + l) * LL + m]; };
    const int ntab = odd ? 3 : 2;
    tab.assign((size_t)ntab * U * NT4, 0.f);
    for (int u = 0; u < U; ++u) {
        const double ct = x[u], st = std::sqrt(1.0 - ct * ct);
        for (int l = 0; l <= LB; ++l)
            for (int m = 0; m <= l; ++m) {
                const double pv = at(u, l, m);
                const size_t k = (size_t)u * NT4 + tri_index(l, m);
                if (l <= p->lmax) {
                    if (!odd) {
                        tab[k] = (float)pv;
                    } else {
                        // d/dtheta P~_lm(cos theta) = (l cos(theta) P~_lm - c_lm P~_(l-1)m) / sin(theta), as in core_host_tables
                        const double pm1 = (l - 1 >= m) ? at(u, l - 1, m) : 0.0;
                        const double c = (l > 0) ? std::sqrt((2.0 * l + 1.0) * ((double)l * l - (double)m * m) / (2.0 * l - 1.0)) : 0.0;
                        tab[k] = (float)((l * ct * pv - c * pm1) / st);
                        tab[(size_t)U * NT4 + k] = (float)(m * pv / st);
                    }
                }
                if (l <= p->lmax_out) tab[(size_t)(ntab - 1) * U * NT4 + k] = (float)(w[u] * pv);
            }
    }
    return NT4;
}

namespace {

struct RegPlan {
    int dev, lmax, lmax_out;
    bool odd;
    int NT4, U, NQ, bytes;
    const void* blob;  // device: even: P[U][NT4], WP[U][NT4]; odd: DP[U][NT4], MP[U][NT4], WP[U][NT4]
    std::vector<float> QF, QI;
};
std::mutex g_mu;
std::vector<RegPlan*> g_plans;

const RegPlan* get_reg_plan(const Plan* p, bool odd)
{
    std::lock_guard<std::mutex> lk(g_mu);
    for (RegPlan* c : g_plans)
        if (c->dev == p->dev && c->lmax == p->lmax && c->lmax_out == p->lmax_out && c->odd == odd) return c;
    std::vector<float> tab;
    const int NT4 = reg_host_tables(p, odd, tab);
    const int U = p->U;
    CoreTab t;
    std::memset(&t, 0, sizeof t);
    std::vector<float> TA, WP, QF, QI;
    core_host_tables(p, odd, t, TA, WP, QF, QI);  // the azimuthal tables of the fast core (quarter-wave rows)
    void* d = nullptr;
    if (cudaMalloc(&d, tab.size() * 4) != cudaSuccess ||
        cudaMemcpy(d, tab.data(), tab.size() * 4, cudaMemcpyHostToDevice) != cudaSuccess) {
        set_error("onsite register core plan: device upload failed: %s", cudaGetErrorString(cudaGetLastError()));
        return nullptr;
    }
    RegPlan* c = new RegPlan;
    c->dev = p->dev;
    c->lmax = p->lmax;
    c->lmax_out = p->lmax_out;
    c->odd = odd;
    c->NT4 = NT4;
    c->U = U;
    c->NQ = t.NQ;
    c->bytes = (int)(tab.size() * 4);
    c->blob = d;
    c->QF = QF;
    c->QI = QI;
    g_plans.push_back(c);
    return c;
}

struct RegArgs {
    const float* tab;
    int tab_floats;
    const float* Ha;
    const float* Hb;
    float* T;
    long long ngroups;
    int U, NQ, L2, Lo2, L2s, Lo2s;
    int off_warp, warp_bytes, off_ts;  // per-warp region: [mbarriers 16 B][H buffers][Ts]
    // two-field coupling (see CoreArgs in onsite_core.cu): factor 2 of edge e is the block of sender send[e]
    const long long* send;
    int cpar;
    const int32_t* status;
};

constexpr int kRegWarps = 4;

template <int LB, bool ODD, bool HREG, int NBUF>
// (register caps for more resident warps at band limits 5 / 6 -- __launch_bounds__(128, 3 or 4): 170 / 128 registers, 200-390
// bytes spilled -- measured slower: lmax 6 odd 111 -> 152 / 119 us, lmax 5 odd 72 -> 78 / 99 us on configs[3])
__global__ void __launch_bounds__(32 * kRegWarps) onsite_reg_kernel(const RegArgs a, const __grid_constant__ CoreQParam<LB> qp)
{
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int NT = (LB + 1) * (LB + 2) / 2, NT4 = round_up(NT, 4), L2B = (LB + 1) * (LB + 1);
    static_assert(!HREG || NBUF == 1, "register-resident H refills its one buffer");
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    pdl_launch_dependents();
    if (a.status) {  // written by an earlier kernel of the stream: nothing may be read before the predecessor is done
        pdl_wait();
        if (*a.status != 0) return;
    }

    float* tabs = reinterpret_cast<float*>(smem);
    for (int i = threadIdx.x; i < a.tab_floats; i += blockDim.x) tabs[i] = a.tab[i];  // the plan's tables: independent
    unsigned char* wr = smem + a.off_warp + (size_t)warp * a.warp_bytes;
    uint64_t* bar = reinterpret_cast<uint64_t*>(wr);  // [NBUF]
    float* hbuf = reinterpret_cast<float*>(wr + 16);
    float* Ts = reinterpret_cast<float*>(wr + a.off_ts);
    const int hfl = 32 * a.L2s;
    const uint32_t hbytes = (uint32_t)hfl * 4;
    if (lane == 0) {
        for (int b = 0; b < NBUF; ++b) mbar_init(&bar[b], 1);
        mbar_fence_init();
    }
    __syncthreads();

    auto load_h = [&](long long g, int buf) {
        float* dst = hbuf + (size_t)buf * 2 * hfl;
        mbar_arrive_expect_tx(&bar[buf], 2 * hbytes);
        tma_load_span(dst, a.Ha + g * hfl, hbytes, &bar[buf]);
        const float* hb = a.Hb + g * hfl;
        if (a.send) {
            const long long c0 = g * 32, e = c0 / a.cpar;
            hb = a.Hb + ((size_t)a.send[e] * a.cpar + (size_t)(c0 - e * a.cpar)) * a.L2s;
        }
        tma_load_span(dst + hfl, hb, hbytes, &bar[buf]);
    };

    const long long stride = (long long)gridDim.x * kRegWarps;
    long long g = (long long)blockIdx.x * kRegWarps + warp;
    pdl_wait();  // H is the predecessor's output
    if (lane == 0 && g < a.ngroups) load_h(g, 0);
    const float* tab0 = tabs;                                   // even: P; odd: d_theta P
    const float* tab1 = tabs + (size_t)a.U * NT4;               // odd: m P / sin(theta)
    const float* tabw = tabs + (size_t)(ODD ? 2 : 1) * a.U * NT4;  // w_u P (analysis)
    int buf = 0;
    uint32_t phases = 0u;
    for (; g < a.ngroups; g += stride) {
        const long long gn = g + stride;
        if (NBUF == 2 && lane == 0 && gn < a.ngroups) load_h(gn, buf ^ 1);
        mbar_wait(&bar[buf], (phases >> buf) & 1u);
        phases ^= 1u << buf;
        const float* ha = hbuf + (size_t)buf * 2 * hfl + lane * a.L2s;
        const float* hb = ha + hfl;
        float2 hh[HREG ? L2B : 1];
        if (HREG) {
#pragma unroll
            for (int k = 0; k < L2B; ++k) hh[k] = (k < a.L2) ? make_float2(ha[k], hb[k]) : make_float2(0.f, 0.f);
            __syncwarp();
            if (lane == 0 && gn < a.ngroups) load_h(gn, 0);  // every lane holds its column: refill the buffer
        }
        float T[L2B];
#pragma unroll
        for (int k = 0; k < L2B; ++k) T[k] = 0.f;

        reg_column_rows<LB, ODD, HREG>(qp, tab0, tab1, tabw, a.U, a.NQ, a.L2, ha, hb, hh, T);

        if (!HREG && NBUF == 1) {  // the rows of H are dead: refill the one buffer while T is stored
            __syncwarp();
            if (lane == 0 && gn < a.ngroups) load_h(gn, 0);
        }
        // ---- T leaves through the warp's staging rows
        if (lane == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
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
        if (NBUF == 2) buf ^= 1;
    }
    if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

template <int LB, bool ODD>
int launch_reg_t(const Plan* p, const RegPlan* c, const float* Ha, const float* Hb, float* T, int64_t ncols, cudaStream_t st,
                 const int64_t* send, int cpar, const int32_t* status)
{
    constexpr bool HREG = LB <= 4;
    constexpr int NBUF = 1;
    RegArgs a;
    a.tab = reinterpret_cast<const float*>(c->blob);
    a.tab_floats = c->bytes / 4;
    a.Ha = Ha;
    a.Hb = Hb;
    a.T = T;
    a.ngroups = (ncols + 31) / 32;  // the caller pads the column count to a multiple of 32
    a.U = c->U;
    a.NQ = c->NQ;
    a.L2 = p->L2;
    a.Lo2 = p->Lo2;
    a.L2s = onsite_fast_hstride(p);
    a.Lo2s = onsite_fast_tstride(p);
    a.send = reinterpret_cast<const long long*>(send);
    a.cpar = cpar;
    a.status = status;
    const int hbytes = 2 * 32 * a.L2s * 4;
    a.off_ts = 16 + NBUF * hbytes;
    a.warp_bytes = round_up(a.off_ts + 32 * a.Lo2s * 4, 128);
    a.off_warp = round_up(c->bytes, 128);
    const size_t smem = (size_t)a.off_warp + (size_t)kRegWarps * a.warp_bytes;
    auto kern = onsite_reg_kernel<LB, ODD, HREG, NBUF>;
    CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int ctas_per_sm = 0;
    CGTP_CUDA_CHECK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas_per_sm, kern, 32 * kRegWarps, smem));
    if (ctas_per_sm < 1) ctas_per_sm = 1;
    int64_t grid = (int64_t)num_sms() * ctas_per_sm;
    const int64_t need = (a.ngroups + kRegWarps - 1) / kRegWarps;
    if (grid > need) grid = need;
    CoreQParam<LB> qp;
    std::memset(&qp, 0, sizeof qp);
    std::memcpy(qp.qf, c->QF.data(), std::min(sizeof qp.qf, c->QF.size() * sizeof(float)));
    std::memcpy(qp.qi, c->QI.data(), std::min(sizeof qp.qi, c->QI.size() * sizeof(float)));
    LaunchScope scope(ODD ? K_ONSITE_ODD : K_ONSITE_EVEN, st);
    CGTP_CUDA_CHECK(launch_pdl(kern, (unsigned)grid, 32u * kRegWarps, smem, st, a, qp));
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

}  // namespace

// Measured on configs[3] (N = C = 32, 16384 atoms; core even / odd in us, this kernel against onsite_fast_kernel):
// lmax 1: 10.5 / 10.7 vs 15.8 / 19.0; 2: 14.8 / 18.9 vs 24.0 / 31.0; 3: 21.0 / 29.1 vs 35.3 / 51.4; 4: 37.3 / 51.7 vs
// 49.7 / 84.4; 5: 55.7 / 72.1 vs 61.9 / 99.0; 6: 100.8 / 110.9 vs 93.0 / 170.4 (223 / 254 registers: 8 warps per SM);
// configs[1] (N = C = 64, 4096 atoms, lmax 6): odd 68.0 vs 88.3.
bool onsite_reg_supported(const Plan* p, bool odd) { return p->LB <= 5 || (p->LB == 6 && odd); }

int launch_onsite_reg(const Plan* p, bool odd, const float* Ha, const float* Hb, float* T, int64_t ncols, cudaStream_t st,
                      const int64_t* send, int cpar, const int32_t* status)
{
    if (ncols <= 0) return CGTP_OK;
    const RegPlan* c = get_reg_plan(p, odd);
    if (!c) return CGTP_ERR_CUDA;
    switch (p->LB) {
#define CGTP_CASE(B)                                                                            \
    case B:                                                                                     \
        return odd ? launch_reg_t<B, true>(p, c, Ha, Hb, T, ncols, st, send, cpar, status)      \
                   : launch_reg_t<B, false>(p, c, Ha, Hb, T, ncols, st, send, cpar, status);
        CGTP_CASE(1) CGTP_CASE(2) CGTP_CASE(3) CGTP_CASE(4) CGTP_CASE(5) CGTP_CASE(6)
#undef CGTP_CASE
    }
    set_error("onsite register core: no kernel for band limit %d", p->LB);
    return CGTP_ERR_UNSUPPORTED;
}

}  // namespace cgtp
