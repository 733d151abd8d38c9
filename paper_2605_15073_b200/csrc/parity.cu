// parity.cu -- routing layer of the parity-slot entry points (Sec. VI :193-:240,
// Sec. VII C a-c, e :383-:469): the index tables that select, for every pass, the weight rows of the runs
// (category, slots, output-l parity sigma) it evaluates, and the kernel that applies Eq.(54)'s restriction
// (-1)^l = sigma to the analysed coefficients.
#include <mutex>
#include <vector>

#include "common.cuh"

namespace cgtp {

// T[col][lm], col = b * Cpar + k: internal channel k belongs to output-l parity tau = (k / Cs) & 1; coefficients of
// the other l-parity are not part of the run (Eq.(54)) and are cleared so that S5 / M6 (Eq.(55), (58))
// sums the two sigma runs of a sector in one contraction.
__global__ void __launch_bounds__(256) sigma_mask_kernel(float* __restrict__ T, int stride, int64_t ncols, int Cpar,
                                                         int Cs, int Lo2)
{
    // one warp per column, lane = lm mod 32: the l-parity of a lane's coefficients is a per-lane bit mask computed
    // once, so the column loop has no division and no square root (32-bit indices: the host rejects ncols >= 2^31)
    const int lane = threadIdx.x & 31;
    uint32_t lodd = 0;  // bit i: degree of lm = lane + 32 i is odd
    for (int lm = lane, i = 0; lm < Lo2; lm += 32, ++i) {
        const int l = (int)sqrtf((float)lm);  // exact: lm < 2^23 and sqrtf is correctly rounded
        lodd |= (uint32_t)(l & 1) << i;
    }
    const uint32_t nwarps = gridDim.x * (blockDim.x >> 5);
    const uint32_t n = (uint32_t)ncols, cpar = (uint32_t)Cpar, cs = (uint32_t)Cs;
    for (uint32_t col = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); col < n; col += nwarps) {
        const uint32_t tau = ((col % cpar) / cs) & 1u;
        const uint32_t clear = tau ? ~lodd : lodd;  // bit i set: coefficient is not part of the run
        float* row = T + (size_t)col * stride;
        for (int lm = lane, i = 0; lm < Lo2; lm += 32, ++i)
            if ((clear >> i) & 1u) row[lm] = 0.f;
    }
}

int launch_sigma_mask(float* T, int stride, int64_t ncols, int Cpar, int Cs, int Lo2, cudaStream_t st)
{
    if (ncols <= 0 || Cpar <= 0) return CGTP_OK;
    if (ncols >= 2147483647LL) { set_error("sigma mask: too many columns"); return CGTP_ERR_UNSUPPORTED; }
    int64_t blocks = (ncols + 7) / 8;
    if (blocks > 148 * 8) blocks = 148 * 8;
    LaunchScope scope(K_MISC, st);
    sigma_mask_kernel<<<(unsigned)blocks, 256, 0, st>>>(T, stride, ncols, Cpar, Cs, Lo2);
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

// ------------------------------------------------------------------------------------------------
// Index tables.  Internal channel order of a pass: [alpha tau=0 | alpha tau=1 | beta tau=0 | beta tau=1], C each;
// the alpha half is the "even" block of the pipeline (pointwise product), the beta half the "odd" block (curl).
//   on-site pass (s1, s2):  run = 8 cat + 4 s1 + 2 s2 + tau          (16 runs, weights [16, C, N] / [16, N, C])
//   message pass s_in:      run = 4 cat + 2 (s_in ^ cat) + tau       ( 8 runs): Eq.(45): alpha reads the slot of
//                           its output sector, Eq.(56): beta the opposite one.
// idx_in[k] = run * C + c (row of the stacked [R*C, N] input weights; column of edge_radial [E, R*C]);
// idx_out[k] = run * N * C + c (offset of the channel inside row n of the stacked W_out; rows are C apart).
// ------------------------------------------------------------------------------------------------
static std::mutex g_pp_mutex;
static std::vector<ParityPlan*> g_pp;

const ParityPlan* get_parity_plan(int C, int N, bool message)
{
    const int ordinal = current_device();
    std::lock_guard<std::mutex> lock(g_pp_mutex);
    for (ParityPlan* q : g_pp)
        if (q->ordinal == ordinal && q->C == C && q->N == N && q->message == message) return q;
    const int npass = message ? 2 : 4;
    std::vector<int> h((size_t)npass * 8 * C);
    for (int ps = 0; ps < npass; ++ps)
        for (int k = 0; k < 4 * C; ++k) {
            const int g = k / C, c = k % C, cat = g >> 1, tau = g & 1;
            const int run = message ? 4 * cat + 2 * (ps ^ cat) + tau : 8 * cat + 4 * (ps >> 1) + 2 * (ps & 1) + tau;
            h[((size_t)ps * 2 + 0) * 4 * C + k] = run * C + c;
            h[((size_t)ps * 2 + 1) * 4 * C + k] = run * N * C + c;
        }
    int* d = nullptr;
    if (cudaMalloc(&d, h.size() * sizeof(int)) != cudaSuccess ||
        cudaMemcpy(d, h.data(), h.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess) {
        set_error("parity plan: device allocation / upload failed");
        return nullptr;
    }
    ParityPlan* q = new ParityPlan;
    q->ordinal = ordinal;
    q->C = C;
    q->N = N;
    q->message = message;
    q->npass = npass;
    q->dev = d;
    g_pp.push_back(q);
    return q;
}

}  // namespace cgtp
