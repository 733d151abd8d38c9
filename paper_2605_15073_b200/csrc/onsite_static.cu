// onsite_static.cu -- cgtp_onsite_static: the on-site contraction S1-S5 (Eq.(35)-(41) PAPER.md:322-346, odd
// channels Eq.(11)-(12) :107-:111) for callers that cannot allocate device memory (CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc).  Every other on-site path of the library keeps the projected coefficients H and the
// rank-space results T in a caller-provided workspace and builds its tables with cudaMalloc on first use; this one
//   * keeps H and T in a FILE-SCOPE device array of kStaticScratchBytes (16 MiB) -- every GPU that loads this module holds
//     it until the process exits --,
//   * passes its (small: band limit <= 4) Legendre and azimuthal tables as kernel parameters, built on the host per call
//     from a host-side cache,
//   * calls no cudaMalloc / cudaFree / allocating library routine, and no plan cache of the library.
// In host code the array's name is a host-side stand-in, not a device address: its address is taken once per device with
// cudaGetSymbolAddress (that device current) and handed to the kernel.
//
// One persistent CTA owns a slot of the array and works on tiles of NA atoms: P (H = W_a . A, W_b . B into the slot) ->
// barrier -> core (one thread per (atom, rank channel) column: reg_column_rows of onsite_reg.cuh, T over the column's
// factor-1 row) -> barrier -> Q (out = W_out . T per sector) -> barrier.  Every word of the slot that a call reads was written
// earlier in the same call by the same CTA, so nothing has to start at zero and the contents left by earlier calls are never
// seen.  ALL CALLS SHARE THE ARRAY: two calls that overlap on the GPU (different streams, or graphs replayed concurrently)
// race on it; calls on one stream are ordered and safe.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <mutex>

#include "cgtp.h"
#include "onsite_reg.cuh"

namespace cgtp {

namespace {

constexpr size_t kStaticScratchBytes = (size_t)16 << 20;
constexpr int kStaticMaxBand = 4;    // max(lmax, lmax_out)
constexpr int kStaticMaxC = 256;     // rank channels
constexpr int kStaticThreads = 256;  // = columns of a tile at most
constexpr int kStaticMaxU = 7;       // ceil((2 lmax + lmax_out + 1) / 2) at band limit 4
constexpr int kStaticTabFloats = 5 * kStaticMaxU * 16;  // even [P][wP], odd [d_theta P][m P / sin][wP], rows of NT4 <= 16

static __device__ __align__(256) float g_static_scratch[kStaticScratchBytes / sizeof(float)];

struct StaticArgs {
    const float *A, *B, *W_a, *W_b, *W_out;
    float* out;
    float* scratch;       // device address of g_static_scratch (cudaGetSymbolAddress)
    long long batch;
    int ntiles, NA;       // atoms per tile: NA * C <= kStaticThreads columns
    int N, C, L2, Lo2, RS;  // RS = row stride of H / T in the slot (odd)
    int U, NQ;
    int slot_floats;      // 2 * NA * C * RS
    unsigned char mask[kStaticMaxC];
    float tab[kStaticTabFloats];
};

template <int LB>
__global__ void __launch_bounds__(kStaticThreads) onsite_static_kernel(const __grid_constant__ StaticArgs a,
                                                                       const __grid_constant__ CoreQParam<LB> qp)
{
    constexpr int NT4 = round_up((LB + 1) * (LB + 2) / 2, 4), L2B = (LB + 1) * (LB + 1);
    __shared__ __align__(16) float tabs[5 * kStaticMaxU * NT4];
    const int tid = threadIdx.x;
    const int N = a.N, C = a.C, L2 = a.L2, Lo2 = a.Lo2, RS = a.RS, U = a.U;
    for (int i = tid; i < 5 * U * NT4; i += kStaticThreads) tabs[i] = a.tab[i];
    const float* te = tabs;                 // even channels: P, w P
    const float* to = tabs + 2 * U * NT4;   // odd channels: d_theta P, m P / sin(theta), w P
    float* Ha = a.scratch + (size_t)blockIdx.x * a.slot_floats;  // this CTA's slot: [NA * C][RS] per factor
    float* Hb = Ha + (size_t)a.NA * C * RS;
    __syncthreads();

    for (int tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
        const long long b0 = (long long)tile * a.NA;
        const int nb = (int)((a.batch - b0 < a.NA) ? (a.batch - b0) : a.NA);
        // ---- P (S1, Eq.(35)): H_f[(at, c)][lm] = sum_n W_f[c][n] X_f[b0 + at][n][lm]
        for (int q = tid; q < 2 * nb * C * L2; q += kStaticThreads) {
            const int lm = q % L2;
            int r = q / L2;
            const int c = r % C;
            r /= C;
            const int at = r % nb, f = r / nb;
            const float* X = (f ? a.B : a.A) + ((size_t)(b0 + at) * N) * L2 + lm;
            const float* W = (f ? a.W_b : a.W_a) + (size_t)c * N;
            float acc = 0.f;
            for (int n = 0; n < N; ++n) acc = fmaf(__ldg(W + n), __ldg(X + (size_t)n * L2), acc);
            (f ? Hb : Ha)[(size_t)(at * C + c) * RS + lm] = acc;
        }
        __syncthreads();
        // ---- core (S2a-S4b): one thread per column, everything on registers; T overwrites the column's factor-1 row
        for (int j = tid; j < nb * C; j += kStaticThreads) {
            float* ha = Ha + (size_t)j * RS;
            const float* hb = Hb + (size_t)j * RS;
            float T[L2B];
#pragma unroll
            for (int k = 0; k < L2B; ++k) T[k] = 0.f;
            const float2 hh[1] = {make_float2(0.f, 0.f)};
            if (a.mask[j % C] == 0)
                reg_column_rows<LB, false, false>(qp, te, te, te + U * NT4, U, a.NQ, L2, ha, hb, hh, T);
            else
                reg_column_rows<LB, true, false>(qp, to, to + U * NT4, to + 2 * U * NT4, U, a.NQ, L2, ha, hb, hh, T);
#pragma unroll
            for (int k = 0; k < L2B; ++k)
                if (k < Lo2) ha[k] = T[k];
        }
        __syncthreads();
        // ---- Q (S5, Eq.(41)): out[b][s][n][lm] = sum_{c: mask[c] = s} W_out[n][c] T[(at, c)][lm]
        for (int q = tid; q < nb * 2 * N * Lo2; q += kStaticThreads) {
            const int lm = q % Lo2;
            int r = q / Lo2;
            const int n = r % N;
            r /= N;
            const int s = r & 1, at = r >> 1;
            const float* W = a.W_out + (size_t)n * C;
            const float* Tr = Ha + (size_t)at * C * RS + lm;
            float acc = 0.f;
            for (int c = 0; c < C; ++c)
                if (a.mask[c] == s) acc = fmaf(__ldg(W + c), Tr[(size_t)c * RS], acc);
            a.out[(((size_t)(b0 + at) * 2 + s) * N + n) * Lo2 + lm] = acc;
        }
        __syncthreads();  // the slot is rewritten by the next tile's P
    }
}

// Host-side table cache (host memory only): per (lmax, lmax_out) the row tables of both parities and the azimuthal tables.
struct StaticTabs {
    int lmax, lmax_out, LB, U, NQ;
    std::vector<float> tab, QF, QI;
};
std::mutex g_mu;
std::vector<StaticTabs*> g_tabs;
float* g_scratch_ptr[64] = {};  // per device ordinal: device address of g_static_scratch

const StaticTabs* get_tabs(int lmax, int lmax_out)
{
    std::lock_guard<std::mutex> lk(g_mu);
    for (StaticTabs* t : g_tabs)
        if (t->lmax == lmax && t->lmax_out == lmax_out) return t;
    Plan p;  // host-side description of the grid only: no device tables, no plan cache of the library
    std::memset(&p, 0, sizeof p);
    p.lmax = lmax;
    p.lmax_out = lmax_out;
    p.nu = 2;
    p.LB = kernel_band(lmax > lmax_out ? lmax : lmax_out);
    p.U = (2 * lmax + lmax_out + 2) / 2;  // ceil((2 lmax + lmax_out + 1) / 2), PAPER.md:173 / DESIGN.md R8
    p.V = 2 * lmax + lmax_out + 1;
    p.Uh = (p.U + 1) / 2;
    p.Vh = p.V / 2 + 1;
    p.L2 = (lmax + 1) * (lmax + 1);
    p.Lo2 = (lmax_out + 1) * (lmax_out + 1);
    StaticTabs* t = new StaticTabs;
    t->lmax = lmax; t->lmax_out = lmax_out; t->LB = p.LB; t->U = p.U;
    std::vector<float> te, to;
    reg_host_tables(&p, false, te);
    reg_host_tables(&p, true, to);
    t->tab = te;
    t->tab.insert(t->tab.end(), to.begin(), to.end());
    CoreTab ct;
    std::memset(&ct, 0, sizeof ct);
    std::vector<float> TA, WP;
    core_host_tables(&p, false, ct, TA, WP, t->QF, t->QI);
    t->NQ = ct.NQ;
    g_tabs.push_back(t);
    return t;
}

template <int LB>
int launch_static_t(const StaticArgs& a, const StaticTabs* t, int grid, cudaStream_t st)
{
    CoreQParam<LB> qp;
    std::memset(&qp, 0, sizeof qp);
    std::memcpy(qp.qf, t->QF.data(), std::min(sizeof qp.qf, t->QF.size() * sizeof(float)));
    std::memcpy(qp.qi, t->QI.data(), std::min(sizeof qp.qi, t->QI.size() * sizeof(float)));
    onsite_static_kernel<LB><<<grid, kStaticThreads, 0, st>>>(a, qp);
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

}  // namespace

}  // namespace cgtp

using namespace cgtp;

extern "C" int cgtp_onsite_static(const float* A, const float* B, const float* W_a, const float* W_b, const float* W_out,
                                  int lmax, int lmax_out, int N, int C, const uint8_t* parity_mask, float* out,
                                  int64_t batch, void* cuda_stream)
{
    clear_error();
    if (lmax < 0 || lmax_out < 0 || lmax_out > 2 * lmax) {
        set_error("invalid band limits lmax=%d lmax_out=%d (need 0 <= lmax_out <= 2*lmax)", lmax, lmax_out);
        return CGTP_ERR_INVALID;
    }
    if (N <= 0 || C <= 0) { set_error("N and C must be positive (N=%d, C=%d)", N, C); return CGTP_ERR_INVALID; }
    if ((lmax > lmax_out ? lmax : lmax_out) > kStaticMaxBand || C > kStaticMaxC) {
        set_error("cgtp_onsite_static: max(lmax,lmax_out)=%d / C=%d exceed the limits of the static scratch array "
                  "(band limit %d, C %d, %zu bytes); use cgtp_onsite with a workspace",
                  lmax > lmax_out ? lmax : lmax_out, C, kStaticMaxBand, kStaticMaxC, kStaticScratchBytes);
        return CGTP_ERR_UNSUPPORTED;
    }
    if (!parity_mask) { set_error("parity_mask is NULL"); return CGTP_ERR_INVALID; }
    for (int c = 0; c < C; ++c)
        if (parity_mask[c] > 1) { set_error("parity_mask[%d]=%d is not 0 or 1", c, (int)parity_mask[c]); return CGTP_ERR_INVALID; }
    if (batch < 0) { set_error("negative batch"); return CGTP_ERR_INVALID; }
    if (batch == 0) return CGTP_OK;
    if (!A || !B || !W_a || !W_b || !W_out || !out) { set_error("null pointer argument"); return CGTP_ERR_INVALID; }

    // device address of the scratch array: once per device, with that device current
    const int dev = current_device();
    if (dev < 0 || dev >= 64) { set_error("cgtp_onsite_static: no current CUDA device"); return CGTP_ERR_CUDA; }
    float* scratch = nullptr;
    {
        std::lock_guard<std::mutex> lk(g_mu);
        if (!g_scratch_ptr[dev]) {
            void* ptr = nullptr;
            const cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_scratch);
            if (e != cudaSuccess || !ptr) {
                set_error("cudaGetSymbolAddress(g_static_scratch) failed: %s", cudaGetErrorString(e));
                return CGTP_ERR_CUDA;
            }
            g_scratch_ptr[dev] = static_cast<float*>(ptr);
        }
        scratch = g_scratch_ptr[dev];
    }
    const StaticTabs* t = get_tabs(lmax, lmax_out);
    if (t->U > kStaticMaxU || (int)t->tab.size() > kStaticTabFloats) {
        set_error("cgtp_onsite_static: table of %zu floats exceeds the kernel parameter block", t->tab.size());
        return CGTP_ERR_UNSUPPORTED;
    }

    StaticArgs a;
    std::memset(&a, 0, sizeof a);
    a.A = A; a.B = B; a.W_a = W_a; a.W_b = W_b; a.W_out = W_out;
    a.out = out;
    a.scratch = scratch;
    a.batch = batch;
    a.N = N; a.C = C;
    a.L2 = (lmax + 1) * (lmax + 1);
    a.Lo2 = (lmax_out + 1) * (lmax_out + 1);
    a.RS = (a.L2 > a.Lo2 ? a.L2 : a.Lo2) | 1;
    a.U = t->U;
    a.NQ = t->NQ;
    a.NA = std::max(1, kStaticThreads / C);
    if ((int64_t)a.NA > batch) a.NA = (int)batch;
    a.slot_floats = 2 * a.NA * C * a.RS;
    const int64_t ntiles = (batch + a.NA - 1) / a.NA;
    if (ntiles > 2147483647LL) { set_error("cgtp_onsite_static: batch too large"); return CGTP_ERR_UNSUPPORTED; }
    a.ntiles = (int)ntiles;
    std::memcpy(a.mask, parity_mask, (size_t)C);
    std::memcpy(a.tab, t->tab.data(), t->tab.size() * sizeof(float));
    // persistent CTAs: two per SM, no more than there are tiles or slots in the array
    int64_t grid = std::min<int64_t>((int64_t)2 * num_sms(), ntiles);
    grid = std::min<int64_t>(grid, (int64_t)(kStaticScratchBytes / sizeof(float)) / a.slot_floats);
    if (grid < 1) { set_error("cgtp_onsite_static: one tile does not fit the static scratch array"); return CGTP_ERR_UNSUPPORTED; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    switch (t->LB) {
        case 1: return launch_static_t<1>(a, t, (int)grid, st);
        case 2: return launch_static_t<2>(a, t, (int)grid, st);
        case 3: return launch_static_t<3>(a, t, (int)grid, st);
        case 4: return launch_static_t<4>(a, t, (int)grid, st);
    }
    set_error("cgtp_onsite_static: no kernel for band limit %d", t->LB);
    return CGTP_ERR_UNSUPPORTED;
}
