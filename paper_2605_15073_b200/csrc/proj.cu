// proj.cu -- channel projections (rows S1, S5, M1, M6 of SURVEY.md 8(a)):
//   Eq.(35)  H[b,c,lm]   = sum_n W[c,n] A[b,n,lm]
//   Eq.(41)  out[b,n,lm] = sum_c W_out[n,c] T[b,c,lm]
//   Eq.(47) (:398), Eq.(55)/(58) (:427,:447) for message passing.
// FP32-exact path: a register-tiled SIMT GEMM whose long dimension is the flattened
// (atom, lm) index, so tiles never need to align with atoms.  The weight matrix is the small
// operand (broadcast from shared memory), the feature matrix is streamed once.
#include "common.cuh"

namespace cgtp {

struct ProjArgPack {
    ProjArgs a[2];
};

constexpr int PROJ_KC = 16;

template <int TM, int TN, int WY>
__global__ void __launch_bounds__(32 * WY) proj_kernel(ProjArgPack pack)
{
    constexpr int NT = 32 * WY;
    constexpr int CW = 32 * TN;   // flattened columns per CTA
    constexpr int MW = WY * TM;   // output rows per CTA
    constexpr int KC = PROJ_KC;
    __shared__ __align__(16) float Xs[KC][CW];
    __shared__ __align__(16) float Ws[KC][MW];

    const ProjArgs a = (blockIdx.z == 0) ? pack.a[0] : pack.a[1];
    const int64_t total = a.batch * (int64_t)a.J;
    const int64_t col0 = (int64_t)blockIdx.x * CW;
    const int m0 = blockIdx.y * MW;
    if (col0 >= total || m0 >= a.M) return;

    const int tid = threadIdx.x, lane = tid & 31, wy = tid >> 5;

    // columns this thread stages into shared memory
    constexpr int NSTG = CW / NT;
    int64_t xbase[NSTG];
#pragma unroll
    for (int i = 0; i < NSTG; ++i) {
        int64_t jj = col0 + tid + i * NT;
        if (jj < total) {
            int64_t b = jj / a.J;
            int j = (int)(jj - b * a.J);
            xbase[i] = b * a.x_bs + j;
        } else {
            xbase[i] = -1;
        }
    }

    float acc[TM][TN];
#pragma unroll
    for (int r = 0; r < TM; ++r)
#pragma unroll
        for (int t = 0; t < TN; ++t) acc[r][t] = 0.f;

    for (int k0 = 0; k0 < a.K; k0 += KC) {
#pragma unroll
        for (int i = 0; i < NSTG; ++i) {
            const int c = tid + i * NT;
#pragma unroll
            for (int kk = 0; kk < KC; ++kk) {
                float v = 0.f;
                if (xbase[i] >= 0 && k0 + kk < a.K) v = __ldg(a.X + xbase[i] + (int64_t)(k0 + kk) * a.x_rs);
                Xs[kk][c] = v;
            }
        }
        for (int idx = tid; idx < KC * MW; idx += NT) {
            const int kk = idx / MW, ml = idx - kk * MW;
            const int m = m0 + ml, k = k0 + kk;
            float v = 0.f;
            if (m < a.M && k < a.K) {
                const int im = a.idx_m ? __ldg(a.idx_m + m) : m;
                const int ik = a.idx_k ? __ldg(a.idx_k + k) : k;
                v = __ldg(a.W + (int64_t)im * a.ldw_m + (int64_t)ik * a.ldw_k);
            }
            Ws[kk][ml] = v;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < KC; ++kk) {
            float w[TM], x[TN];
#pragma unroll
            for (int r = 0; r < TM; r += 4) {
                float4 t4 = *reinterpret_cast<const float4*>(&Ws[kk][wy * TM + r]);
                w[r] = t4.x; w[r + 1] = t4.y; w[r + 2] = t4.z; w[r + 3] = t4.w;
            }
#pragma unroll
            for (int t = 0; t < TN; ++t) x[t] = Xs[kk][lane + 32 * t];
#pragma unroll
            for (int r = 0; r < TM; ++r)
#pragma unroll
                for (int t = 0; t < TN; ++t) acc[r][t] = fmaf(w[r], x[t], acc[r][t]);
        }
        __syncthreads();
    }

#pragma unroll
    for (int t = 0; t < TN; ++t) {
        const int64_t jj = col0 + lane + 32 * t;
        if (jj >= total) continue;
        const int64_t b = jj / a.J;
        const int j = (int)(jj - b * a.J);
#pragma unroll
        for (int r = 0; r < TM; ++r) {
            const int m = m0 + wy * TM + r;
            if (m >= a.M) continue;
            float* dst = (m < a.m_split) ? a.out0 + b * a.o_bs0 + (int64_t)m * a.o_rs + j
                                         : a.out1 + b * a.o_bs1 + (int64_t)(m - a.m_split) * a.o_rs + j;
            *dst = a.accumulate ? *dst + acc[r][t] : acc[r][t];
        }
    }
}

// A problem with an empty contraction (K == 0: a parity sector without rank channels) has an all-zero result.
// When its output rows are one dense block per batch entry it is written by a 2-D memset, so that the remaining
// problem keeps the fast kernels; returns false when the layout is not of that form.
static bool zero_fill(const ProjArgs& g, cudaStream_t st, int* rc)
{
    *rc = CGTP_OK;
    if (g.batch <= 0 || g.M <= 0 || g.J <= 0 || g.accumulate) return true;  // adding zero: nothing to do
    if (g.o_rs != g.J || g.m_split < g.M) return false;
    const cudaError_t e = cudaMemset2DAsync(g.out0, (size_t)g.o_bs0 * 4, 0, (size_t)g.M * g.J * 4, (size_t)g.batch, st);
    if (e != cudaSuccess) {
        set_error("cudaMemset2DAsync failed: %s", cudaGetErrorString(e));
        *rc = CGTP_ERR_CUDA;
    }
    return true;
}

int launch_proj(const ProjArgs* args_in, int nargs_in, Kind kind, cudaStream_t st)
{
    if (nargs_in < 1 || nargs_in > 2) { set_error("launch_proj: nargs"); return CGTP_ERR_INVALID; }
    ProjArgs kept[2];
    int nargs = 0;
    for (int i = 0; i < nargs_in; ++i) {
        int rc = CGTP_OK;
        if (args_in[i].K == 0 && zero_fill(args_in[i], st, &rc)) {
            if (rc != CGTP_OK) return rc;
            continue;
        }
        kept[nargs++] = args_in[i];
    }
    if (nargs == 0) return CGTP_OK;
    const ProjArgs* args = kept;
    ProjArgPack pack;
    int64_t max_cols = 0;
    int max_m = 0;
    for (int i = 0; i < nargs; ++i) {
        pack.a[i] = args[i];
        int64_t cols = args[i].batch * (int64_t)args[i].J;
        if (cols > max_cols) max_cols = cols;
        if (args[i].M > max_m) max_m = args[i].M;
    }
    if (nargs == 1) pack.a[1] = args[0];
    if (max_cols == 0 || max_m == 0) return CGTP_OK;
    bool offset = false;
    for (int i = 0; i < nargs; ++i) offset = offset || args[i].j0 != 0;
    if (!offset) {
        bool handled = false;
        const int rc = launch_proj_tc(args, nargs, kind, st, &handled);
        if (rc != CGTP_OK || handled) return rc;
    }
    if (!(kernel_path() & PATH_GENERIC_PROJ)) {
        bool handled = false;
        const int rc = launch_proj_fast(args, nargs, kind, st, &handled);
        if (rc != CGTP_OK || handled) return rc;
    }
    for (int i = 0; i < 2; ++i) {  // the generic kernel loads scalars: fold the column offset into the pointer
        pack.a[i].X += pack.a[i].j0;
        pack.a[i].j0 = 0;
    }
    constexpr int TM = 8, TN = 8;
    const int CW = 32 * TN;
    int64_t gx = (max_cols + CW - 1) / CW;
    if (gx > 2147483647LL) { set_error("launch_proj: too many columns"); return CGTP_ERR_UNSUPPORTED; }
    LaunchScope scope(kind, st);
    if (max_m <= 32) {
        constexpr int WY = 4;
        dim3 grid((unsigned)gx, (max_m + WY * TM - 1) / (WY * TM), nargs);
        proj_kernel<TM, TN, WY><<<grid, 32 * WY, 0, st>>>(pack);
    } else {
        constexpr int WY = 8;
        dim3 grid((unsigned)gx, (max_m + WY * TM - 1) / (WY * TM), nargs);
        proj_kernel<TM, TN, WY><<<grid, 32 * WY, 0, st>>>(pack);
    }
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

}  // namespace cgtp
