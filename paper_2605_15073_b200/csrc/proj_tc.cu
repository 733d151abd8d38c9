// proj_tc.cu -- tensor-core variants of the channel projections (rows S1, S5, M1, M6 of SURVEY.md 8(a);
// Eq.(35), Eq.(41) :346, Eq.(47) :398, Eq.(55)/(58) :427,:447) on the 5th-generation
// tensor cores: tcgen05.mma kind::tf32, accumulators in tensor memory (TMEM).  Selected by
// cgtp_set_math_mode (1 = 3xTF32, 2 = TF32); never the default: the FP32-exact path is proj_fast.cu.
//
// GEMM orientation.  D[col, c] = sum_k Xt[col, k] W[c, k] with col the flattened (atom, lm) index:
//   A operand = X^T tile, 128 columns x KC, K-major;  B operand = W, Npad channels x KC, K-major;
//   D = 128 TMEM lanes (one per column) x Npad TMEM columns (one per output channel), FP32.
// So the epilogue thread of lane r owns one output column and, channel by channel, a warp writes 32
// consecutive lm of one output row: coalesced 128-byte stores.
//
// Shared-memory operand layout: the canonical no-swizzle K-major layout of the UMMA descriptor (core
// matrix = 8 rows x 16 bytes, rows 16 B apart; 8-row groups SBO = 128 B apart; the two 16-byte K halves
// of one K = 8 instruction LBO apart) -- i.e. a float4 array [k/4][row].  X has lm contiguous and odd row
// lengths, so no TMA tensor map fits it: loader threads read 4 consecutive k of one column with
// coalesced 32-bit loads and write one 128-bit element of the array (transpose on the fly).
//
// 3xTF32: x = hi + lo with hi = the 19 leading bits the tensor core reads, lo = x - hi (exact in FP32);
// D = A_hi B_lo + A_lo B_hi + A_hi B_hi accumulated in FP32 in TMEM; the dropped lo*lo term and the
// truncation of lo are ~2^-21 relative per product.  TF32: the A_hi B_hi term alone (~2^-10).
//
// Roles (544 threads): warps 0-7 epilogue (TMEM lane quarter = warp index % 4), warps 8-15 loaders,
// warp 16 issues the MMAs (one elected thread).  Two shared-memory stages and two TMEM accumulators
// are linked by mbarriers (tcgen05.commit arrives on them when the MMAs that read a stage finish).
#include <algorithm>

#include "sht.cuh"

namespace cgtp {

constexpr int TC_COLS = 128;     // columns per tile = UMMA M
constexpr int TC_EPI_WARPS = 8;   // two warps per TMEM lane quarter, each takes alternate 32-channel slices
constexpr int TC_LD_WARPS = 8;
constexpr int TC_THREADS = 32 * (TC_EPI_WARPS + TC_LD_WARPS + 1);
constexpr int TC_STAGES = 2;

struct TcProblem {
    const float* X;
    int64_t x_bs;
    int x_rs;
    const float* W;
    int ldw_m, ldw_k;
    const int* idx_m;
    const int* idx_k;
    int M, K;  // output channels, contraction length
    float* out0;
    int64_t o_bs0;
    float* out1;
    int64_t o_bs1;
    int m_split;
    int o_rs;
    int cta_begin, ctas;
};

struct TcArgs {
    TcProblem p[2];
    int nprob;
    int J;
    int64_t batch;
    int Npad;      // channels padded to a multiple of 16 (UMMA N)
    int Kpad;      // max K padded to a multiple of KC
    int KC;        // contraction chunk per stage (multiple of 8)
    int split;     // 1: 3xTF32 (hi/lo operands), 0: single TF32
    int tmem_cols; // power of two >= 2*Npad, >= 32
};

// ---------------------------------------------------------------------------------- tcgen05 wrappers
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void tc_mma_tf32(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc, uint32_t acc)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(acc)
        : "memory");
}
__device__ __forceinline__ void tc_commit(uint64_t* bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive1(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// K-major, no swizzle: start address, leading (K-half) and stride (8-row group) byte offsets, version 1.
__device__ __forceinline__ uint64_t tc_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo)
{
    return (uint64_t)((saddr >> 4) & 0x3fffu) | ((uint64_t)((lbo >> 4) & 0x3fffu) << 16) |
           ((uint64_t)((sbo >> 4) & 0x3fffu) << 32) | (1ull << 46);
}
// 32 lanes x 32 consecutive TMEM columns -> 32 registers per thread
__device__ __forceinline__ void tc_ld32(uint32_t taddr, uint32_t (&v)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
        "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
          "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
          "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

__device__ __forceinline__ float tf32_hi(float x) { return __uint_as_float(__float_as_uint(x) & 0xffffe000u); }

template <bool ACC>
__global__ void __launch_bounds__(TC_THREADS, 1) proj_tc_kernel(TcArgs a)
{
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);       // [TC_STAGES]  loaders -> MMA
    uint64_t* empty = full + TC_STAGES;                        // [TC_STAGES]  MMA -> loaders
    uint64_t* tfull = empty + TC_STAGES;                       // [2]          MMA -> epilogue
    uint64_t* tempty = tfull + 2;                              // [2]          epilogue -> MMA
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + 2);
    const int Npad = a.Npad, KC = a.KC, KG = KC / 4;
    const int nsplit = a.split ? 2 : 1;
    // W: [nsplit][Kpad/4][Npad] float4;  stages: [TC_STAGES][nsplit][KG][128] float4
    float4* Ws = reinterpret_cast<float4*>(smem + 128);
    const int w_f4 = (a.Kpad / 4) * Npad;
    float4* As = Ws + (size_t)nsplit * w_f4;
    const int a_f4 = KG * TC_COLS;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int pi = (a.nprob > 1 && (int)blockIdx.x >= a.p[1].cta_begin) ? 1 : 0;
    const TcProblem& P = a.p[pi];
    const int rank = blockIdx.x - P.cta_begin, nctas = P.ctas;
    const int K = P.K, M = P.M;
    const int NCH = (K + KC - 1) / KC;
    const int64_t total_cols = a.batch * (int64_t)a.J;
    const int64_t ntiles = (total_cols + TC_COLS - 1) / TC_COLS;

    if (tid == 0) {
        for (int s = 0; s < TC_STAGES; ++s) {
            mbar_init(&full[s], TC_LD_WARPS);
            mbar_init(&empty[s], 1);
        }
        for (int s = 0; s < 2; ++s) {
            mbar_init(&tfull[s], 1);
            mbar_init(&tempty[s], TC_EPI_WARPS);
        }
        mbar_fence_init();
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)),
                     "r"((uint32_t)a.tmem_cols)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    // weights -> canonical K-major layout, split into hi / lo; rows >= M and k >= K are zero
    for (int idx = tid; idx < w_f4; idx += TC_THREADS) {
        const int kg = idx / Npad, n = idx - kg * Npad;
        float v[4] = {0.f, 0.f, 0.f, 0.f};
        if (n < M) {
            const int im = P.idx_m ? __ldg(P.idx_m + n) : n;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int k = 4 * kg + q;
                if (k < K) {
                    const int ik = P.idx_k ? __ldg(P.idx_k + k) : k;
                    v[q] = __ldg(P.W + (int64_t)im * P.ldw_m + (int64_t)ik * P.ldw_k);
                }
            }
        }
        if (a.split) {
            const float4 hi = make_float4(tf32_hi(v[0]), tf32_hi(v[1]), tf32_hi(v[2]), tf32_hi(v[3]));
            Ws[idx] = hi;
            Ws[w_f4 + idx] = make_float4(v[0] - hi.x, v[1] - hi.y, v[2] - hi.z, v[3] - hi.w);
        } else {
            Ws[idx] = make_float4(v[0], v[1], v[2], v[3]);
        }
    }
    fence_async_smem();  // generic-proxy writes of W -> visible to the tensor core (async proxy)
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp >= TC_EPI_WARPS && warp < TC_EPI_WARPS + TC_LD_WARPS) {
        // ======================================= loaders =======================================
        const int lt = tid - 32 * TC_EPI_WARPS;       // 0..255
        const int col = lt & (TC_COLS - 1);            // column of the tile
        const int half = lt >> 7;                      // which half of the chunk's k-groups
        const int kg_begin = half * (KG / 2), kg_end = (half + 1) * (KG / 2);
        // unit = (tile, K chunk).  The loads of the next unit are issued before the current one is stored, so a
        // thread keeps up to 2 x 32 independent 32-bit loads in flight (register double buffering).
        auto load_unit = [&](int64_t t, int ch, float (&v)[8][4]) {
            const int64_t cc = t * TC_COLS + col;
            const bool live = cc < total_cols;
            const int64_t b = live ? cc / a.J : 0;
            const int j = live ? (int)(cc - b * a.J) : 0;
            const float* xcol = P.X + b * P.x_bs + j;
#pragma unroll
            for (int g = 0; g < 8; ++g)
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const int k = ch * KC + 4 * (kg_begin + g) + q;
                    v[g][q] = (live && kg_begin + g < kg_end && k < K) ? __ldg(xcol + (int64_t)k * P.x_rs) : 0.f;
                }
        };
        int s = 0;
        uint32_t ph = 0;
        float cur[8][4], nxt[8][4];
        int64_t t = rank;
        int ch = 0;
        if (t < ntiles) load_unit(t, ch, cur);
        while (t < ntiles) {
            int64_t tn = t;
            int chn = ch + 1;
            if (chn == NCH) { chn = 0; tn += nctas; }
            if (tn < ntiles) load_unit(tn, chn, nxt);
            mbar_wait(&empty[s], ph ^ 1u);
            float4* dst_hi = As + (size_t)s * nsplit * a_f4;
            float4* dst_lo = dst_hi + a_f4;
#pragma unroll
            for (int g = 0; g < 8; ++g) {
                if (kg_begin + g >= kg_end) break;
                const int di = (kg_begin + g) * TC_COLS + col;
                if (a.split) {
                    const float4 hi = make_float4(tf32_hi(cur[g][0]), tf32_hi(cur[g][1]), tf32_hi(cur[g][2]), tf32_hi(cur[g][3]));
                    dst_hi[di] = hi;
                    dst_lo[di] = make_float4(cur[g][0] - hi.x, cur[g][1] - hi.y, cur[g][2] - hi.z, cur[g][3] - hi.w);
                } else {
                    dst_hi[di] = make_float4(cur[g][0], cur[g][1], cur[g][2], cur[g][3]);
                }
            }
            fence_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive1(&full[s]);
            if (++s == TC_STAGES) { s = 0; ph ^= 1u; }
#pragma unroll
            for (int g = 0; g < 8; ++g)
#pragma unroll
                for (int q = 0; q < 4; ++q) cur[g][q] = nxt[g][q];
            t = tn;
            ch = chn;
        }
    } else if (warp == TC_EPI_WARPS + TC_LD_WARPS) {
        // ======================================= MMA issuer =====================================
        if (lane == 0) {
            // instruction descriptor: D = F32, A = B = TF32, both K-major, N = Npad, M = 128
            const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(Npad >> 3) << 17) | ((uint32_t)(TC_COLS >> 4) << 24);
            const uint32_t w_base = smem_u32(Ws), a_base = smem_u32(As);
            const uint32_t lbo_a = TC_COLS * 16, lbo_b = (uint32_t)Npad * 16;
            int s = 0, acc = 0;
            uint32_t ph = 0, aph = 0;
            for (int64_t t = rank; t < ntiles; t += nctas) {
                mbar_wait(&tempty[acc], aph ^ 1u);
                tc_fence_after();
                const uint32_t d = tmem_base + (uint32_t)(acc * Npad);
                uint32_t accum = 0;
                for (int ch = 0; ch < NCH; ++ch) {
                    mbar_wait(&full[s], ph);
                    tc_fence_after();
                    const uint32_t a_hi = a_base + (uint32_t)(s * nsplit * a_f4) * 16u;
                    const uint32_t a_lo = a_hi + (uint32_t)a_f4 * 16u;
                    const uint32_t b_hi = w_base + (uint32_t)(ch * KG * Npad) * 16u;
                    const uint32_t b_lo = b_hi + (uint32_t)w_f4 * 16u;
                    for (int ks = 0; ks < KC / 8; ++ks) {
                        const uint32_t ao = (uint32_t)(2 * ks) * lbo_a, bo = (uint32_t)(2 * ks) * lbo_b;
                        if (a.split) {
                            tc_mma_tf32(d, tc_desc(a_hi + ao, lbo_a, 128), tc_desc(b_lo + bo, lbo_b, 128), idesc, accum);
                            tc_mma_tf32(d, tc_desc(a_lo + ao, lbo_a, 128), tc_desc(b_hi + bo, lbo_b, 128), idesc, 1u);
                            accum = 1u;
                        }
                        tc_mma_tf32(d, tc_desc(a_hi + ao, lbo_a, 128), tc_desc(b_hi + bo, lbo_b, 128), idesc, accum);
                        accum = 1u;
                    }
                    tc_commit(&empty[s]);  // the stage may be refilled once these MMAs have read it
                    if (++s == TC_STAGES) { s = 0; ph ^= 1u; }
                }
                tc_commit(&tfull[acc]);
                if (++acc == 2) { acc = 0; aph ^= 1u; }
            }
        }
    } else if (warp < TC_EPI_WARPS) {
        // ======================================= epilogue =======================================
        int acc = 0;
        uint32_t aph = 0;
        const int quarter = warp & 3, slice0 = warp >> 2;  // TMEM lanes 32*quarter..+31; channel slices slice0, slice0+2, ..
        const int o_rs = P.o_rs, m_split = P.m_split;
        for (int64_t t = rank; t < ntiles; t += nctas) {
            const int64_t cc = t * TC_COLS + 32 * quarter + lane;
            const bool live = cc < total_cols;
            const int64_t b = live ? cc / a.J : 0;
            const int j = live ? (int)(cc - b * a.J) : 0;
            float* o0 = P.out0 + b * P.o_bs0 + j;
            float* o1 = P.out1 + b * P.o_bs1 + j - (int64_t)m_split * o_rs;
            mbar_wait(&tfull[acc], aph);
            tc_fence_after();
            const uint32_t taddr = tmem_base + ((uint32_t)(32 * quarter) << 16) + (uint32_t)(acc * Npad);
            for (int c0 = 32 * slice0; c0 < M; c0 += 32 * (TC_EPI_WARPS / 4)) {
                uint32_t v[32];
                tc_ld32(taddr + (uint32_t)c0, v);
                if (live) {
                    if (c0 + 32 <= m_split || c0 >= m_split) {  // the whole slice goes to one output tensor
                        float* p = ((c0 < m_split) ? o0 : o1) + (int64_t)c0 * o_rs;
                        const int nq = (M - c0 < 32) ? (M - c0) : 32;
                        if (ACC) {
                            // all loads before the first store (a load behind a possibly aliasing store waits for it)
#pragma unroll
                            for (int q = 0; q < 32; ++q)
                                if (q < nq) v[q] = __float_as_uint(__uint_as_float(v[q]) + __ldcg(p + (int64_t)q * o_rs));
                        }
#pragma unroll
                        for (int q = 0; q < 32; ++q) {
                            if (q < nq) *p = __uint_as_float(v[q]);
                            p += o_rs;
                        }
                    } else {
#pragma unroll
                        for (int q = 0; q < 32; ++q) {
                            const int m = c0 + q;
                            if (m < M) {
                                float* w = ((m < m_split) ? o0 : o1) + (int64_t)m * o_rs;
                                *w = ACC ? *w + __uint_as_float(v[q]) : __uint_as_float(v[q]);
                            }
                        }
                    }
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive1(&tempty[acc]);
            if (++acc == 2) { acc = 0; aph ^= 1u; }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 0) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"((uint32_t)a.tmem_cols)
                     : "memory");
    }
}

// ------------------------------------------------------------------------------------------------
// Host
// ------------------------------------------------------------------------------------------------
static int g_math_mode = 0;
void set_math_mode(int m) { g_math_mode = m; }
int get_math_mode() { return g_math_mode; }


// *handled = false: not in a tensor-core math mode, or the shapes do not fit (caller uses the FP32 kernels).
int launch_proj_tc(const ProjArgs* args, int nargs, Kind kind, cudaStream_t st, bool* handled)
{
    *handled = false;
    if (g_math_mode == 0 || nargs < 1 || nargs > 2) return CGTP_OK;
    const int J = args[0].J;
    const int64_t batch = args[0].batch;
    int maxM = 0, maxK = 0;
    for (int i = 0; i < nargs; ++i) {
        if (args[i].J != J || args[i].batch != batch || args[i].M < 1 || args[i].K < 1 ||
            args[i].accumulate != args[0].accumulate)
            return CGTP_OK;
        maxM = std::max(maxM, args[i].M);
        maxK = std::max(maxK, args[i].K);
    }
    if (batch <= 0 || J <= 0) return CGTP_OK;
    const int split = (g_math_mode == 1) ? 1 : 0;
    const int nsplit = split ? 2 : 1;
    // the TMEM lane quarter a warp may read holds 32 columns x Npad channels; the epilogue reads 32-column
    // slices, so channels are padded to a multiple of 32
    const int Npad = round_up(maxM, 32);
    if (Npad > 256) return CGTP_OK;
    int tmem_cols = 32;
    while (tmem_cols < 2 * Npad) tmem_cols <<= 1;
    const size_t budget = 200 * 1024;
    int KC = 0, Kpad = 0;
    for (int kc : {64, 32, 16, 8}) {
        const int kp = round_up(maxK, kc);
        const size_t need = 128 + (size_t)nsplit * kp * Npad * 4 + (size_t)TC_STAGES * nsplit * kc * TC_COLS * 4;
        if (need <= budget) { KC = kc; Kpad = kp; break; }
    }
    if (!KC) return CGTP_OK;

    TcArgs a;
    a.nprob = nargs;
    a.J = J;
    a.batch = batch;
    a.Npad = Npad;
    a.Kpad = Kpad;
    a.KC = KC;
    a.split = split;
    a.tmem_cols = tmem_cols;
    const size_t smem = 128 + (size_t)nsplit * Kpad * Npad * 4 + (size_t)TC_STAGES * nsplit * KC * TC_COLS * 4;
    const int64_t ntiles = (batch * (int64_t)J + TC_COLS - 1) / TC_COLS;
    const int slots = num_sms();
    double wsum = 0.0;
    for (int i = 0; i < nargs; ++i) wsum += args[i].K;
    int begin = 0;
    for (int i = 0; i < nargs; ++i) {
        const ProjArgs& g = args[i];
        TcProblem& q = a.p[i];
        q.X = g.X; q.x_bs = g.x_bs; q.x_rs = g.x_rs; q.W = g.W; q.ldw_m = g.ldw_m; q.ldw_k = g.ldw_k;
        q.idx_m = g.idx_m; q.idx_k = g.idx_k; q.M = g.M; q.K = g.K;
        q.out0 = g.out0; q.o_bs0 = g.o_bs0; q.out1 = g.out1; q.o_bs1 = g.o_bs1; q.m_split = g.m_split; q.o_rs = g.o_rs;
        int n = (int)((double)slots * g.K / wsum);
        if (n < 1) n = 1;
        if ((int64_t)n > ntiles) n = (int)ntiles;
        q.cta_begin = begin;
        q.ctas = n;
        begin += n;
    }
    if (nargs == 1) a.p[1] = a.p[0];

    LaunchScope scope(kind, st);
    void (*kern)(TcArgs) = args[0].accumulate ? proj_tc_kernel<true> : proj_tc_kernel<false>;  // out += result
    CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<begin, TC_THREADS, smem, st>>>(a);
    CGTP_CUDA_CHECK(cudaGetLastError());
    *handled = true;
    return CGTP_OK;
}

}  // namespace cgtp
