// proj_fast.cu -- FP32-exact channel projections (rows S1, S5, M1, M6 of SURVEY.md 8(a); Eq.(35)
// PAPER.md:322, Eq.(41) :346, Eq.(47) :398, Eq.(55)/(58) :427,:447) as a streaming SIMT GEMM built for
// sm_100a:
//   * the feature operand X[b] (K rows of one atom, contiguous in HBM) is staged by TMA bulk copies
//     (cp.async.bulk + mbarrier complete_tx) into a multi-stage shared-memory ring, K-chunk by K-chunk,
//     for a group of AB atoms whose AB*J flattened columns fill the CTA's column window;
//   * the weight tile is loaded once per (persistent) CTA and kept in shared memory as Ws[k][row]; every
//     multiply-add is a packed FFMA2 (fma.rn.f32x2) on a pair of adjacent output rows: a thread owns
//     16 rows x 4 columns = 32 float2 accumulators, the weight pair (w[r],w[r+1]) comes straight from a
//     128-bit broadcast load, the feature value is duplicated in registers.  Per k: 4 LDS.128 + 4 LDS.32
//     for 32 FFMA2 -- 8 shared-memory wavefronts per 64 FMA-pipe cycles.  One CTA of 8 warps per SM with
//     ~230 registers per thread and the K loop unrolled by 8, so that the shared-memory loads of the next
//     steps are in flight under the FFMA2s of the current one (measured: 0.093 ms against 0.105 ms for two
//     CTAs per SM capped at 128 registers, configs[1] S1);
//   * each CTA serves one (problem, row block) for its whole life and strides over atom groups.
// Summation over k runs in ascending order with one accumulator per output, as in proj.cu.
#include <algorithm>

#include "sht.cuh"

namespace cgtp {

constexpr int kPfThreads = 256;

struct PfProblem {
    const float* X;
    int64_t x_bs;
    int x_rs;
    const float* W;
    int ldw_m, ldw_k;
    const int* idx_m;
    const int* idx_k;
    int M, K;
    float* out0;
    int64_t o_bs0;
    float* out1;
    int64_t o_bs1;
    int m_split;
    int o_rs;
    int j0;        // first used column of every X row
    int nrb;       // row blocks of this problem
    int cta_begin; // first CTA (blockIdx.x) serving this problem
    int ctas_per_rb;
};

struct PfArgs {
    PfProblem p[2];
    int nprob;
    int J;
    int64_t batch;
    int AB, KC, NSTAGE, NSUB;
    int stage_floats;  // AB * KC * x_rs
    uint32_t jmagic;   // floor(2^32 / J) + 1
    int w_floats;      // Kmax * MW
    int window;        // 1: tile = window of CWT flattened (atom, j) columns, atoms may straddle tiles (NSUB = 1)
    int ntiles;        // tiles per (problem, row block)
};

__device__ __forceinline__ float lds32(uint32_t addr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ float4 lds128(uint32_t addr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

// store at a compile-time byte offset from a per-thread pointer: STG [R.64 + imm], no address arithmetic per store
template <int OFF>
__device__ __forceinline__ void stg_off(float* p, float v)
{
    asm volatile("st.global.f32 [%0+%1], %2;" ::"l"(p), "n"(OFF), "f"(v) : "memory");
}

__device__ __forceinline__ void mbar_arrive_cta(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// RS > 0: the row strides of X and of the output are both the compile-time constant RS (floats) -- the x loads of the
// inner loop and the stores of the epilogue then address with immediate offsets (no per-load IMAD, no per-store address
// arithmetic: 31 of 363 instructions per 8 k-steps and ~80 of 100 per 16 stores with run-time strides, ncu source
// counters at configs[1]).  RS = 0: run-time strides.
template <int RW, int CWP, bool ACC, bool WIN, int RS = 0>
__global__ void __launch_bounds__(kPfThreads, 1) proj_fast_kernel(PfArgs a)
{
    constexpr int MW = 16 * RW;       // rows per CTA
    constexpr int CWT = 128 * CWP;    // flattened columns per tile
    static_assert(RW * CWP == 8, "8 consumer warps");
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);  // [NSTAGE <= 3]  TMA -> consumers
    uint64_t* empty = full + 4;                          // [NSTAGE]       consumer warps -> producer (warp 0)
    float* Wd = reinterpret_cast<float*>(smem + 64);
    float* stages = Wd + a.w_floats;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wr = warp % RW, wc = warp / RW;

    // which (problem, row block, rank within the row block) this CTA serves; the fields are copied to
    // registers once (indexing the parameter struct at run time would cost a constant load per use)
    const int pi = (a.nprob > 1 && (int)blockIdx.x >= a.p[1].cta_begin) ? 1 : 0;
    const float* const X = pi ? a.p[1].X : a.p[0].X;
    const int64_t x_bs = pi ? a.p[1].x_bs : a.p[0].x_bs;
    const int x_rs = RS ? RS : a.p[0].x_rs;  // common to both problems (host-checked)
    const int M = pi ? a.p[1].M : a.p[0].M;
    const int K = pi ? a.p[1].K : a.p[0].K;
    const int cpr = pi ? a.p[1].ctas_per_rb : a.p[0].ctas_per_rb;
    const int j0 = pi ? a.p[1].j0 : a.p[0].j0;
    const int local = blockIdx.x - (pi ? a.p[1].cta_begin : 0);
    const int rb = local / cpr, rank = local - rb * cpr;
    const int m0 = rb * MW;
    const int J = a.J, AB = a.AB, NSUB = a.NSUB, NSTAGE = a.NSTAGE, KC = a.KC;
    const uint32_t jmagic = a.jmagic;  // cc / J == umulhi(cc, jmagic) for cc < 2^16

    if (tid == 0) {
        for (int s = 0; s < NSTAGE; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], kPfThreads / 32);
        }
        mbar_fence_init();
    }
    __syncthreads();

    // tiles of this CTA: ti = rank + i * cpr (32-bit: the host rejects larger problems); chunk counters
    // advance incrementally (no divisions in the loop)
    // tiles of a (problem, row block): WIN = false: (atom group, sub-tile); WIN = true: windows of CWT flattened
    // (atom, j) columns (NSUB = 1), atoms may straddle tiles.  A template flag so that the group form keeps its code.
    const int ntiles = a.ntiles;
    // first atom of tile ti and the tile's first column inside the staged atoms
    auto tile_origin = [&](int ti, int& b0, int& off0) {
        if (WIN) {
            const int64_t c0 = (int64_t)ti * CWT;
            b0 = (int)(c0 / J);
            off0 = (int)(c0 - (int64_t)b0 * J);
        } else {
            const int g = ti / NSUB;
            b0 = g * AB;
            off0 = (ti - g * NSUB) * CWT;
        }
    };
    const int my_tiles = (ntiles > rank) ? (ntiles - rank + cpr - 1) / cpr : 0;
    const int NCH = K / KC;
    const int nchunks = my_tiles * NCH;
    const int chunk_floats = KC * x_rs;
    const uint32_t chunk_bytes = (uint32_t)chunk_floats * 4u;

    // warp 0 issues the bulk copies of the chunk (tile ti, K-chunk kc) into slot s (lane = atom within the group)
    auto issue = [&](int ti, int kc, int s) {
        int b0, off0;
        tile_origin(ti, b0, off0);
        const int nb = (int)((a.batch - b0 < AB) ? (a.batch - b0) : AB);
        float* dst = stages + (size_t)s * a.stage_floats;
        if (lane == 0) mbar_arrive_expect_tx(&full[s], chunk_bytes * (uint32_t)nb);
        __syncwarp();
        for (int al = lane; al < nb; al += 32)
            tma_load_1d(dst + (size_t)al * chunk_floats, X + ((int64_t)b0 + al) * x_bs + (int64_t)kc * chunk_floats, chunk_bytes,
                        &full[s]);
    };

    // producer cursor (chunk index pc, its tile / K-chunk / slot) runs NSTAGE-1 chunks ahead
    int pc = 0, p_ti = rank, p_kc = 0, p_s = 0;
    auto produce = [&]() {
        if (warp == 0 && pc < nchunks) issue(p_ti, p_kc, p_s);
        ++pc;
        if (++p_kc == NCH) { p_kc = 0; p_ti += cpr; }
        if (++p_s == NSTAGE) p_s = 0;
    };
    // Programmatic dependent launch (common.cuh): this kernel may be scheduled while its predecessor in the stream still
    // runs.  Everything it reads from global memory is a caller input or the predecessor's output (X, and the weights too:
    // the caller's previous kernel may have just written them), so it waits here; what overlaps is the launch itself and
    // the barrier set-up above.
    pdl_launch_dependents();
    pdl_wait();
    for (int i = 0; i < NSTAGE - 1; ++i) produce();

    // ---- weights: Wd[k][r] = W[idx_m[m0+r]][idx_k[k]].  Thread = fixed row r,
    // strided k: the loads of different k are independent and stay in flight together.
    {
        const PfProblem& P = a.p[pi];
        constexpr int KSTEP = kPfThreads / MW;
        const int r = tid % MW, kq = tid / MW;
        const int m = m0 + r;
        const bool live = m < M;
        const int im = live ? (P.idx_m ? __ldg(P.idx_m + m) : m) : 0;
        const float* wsrc = P.W + (int64_t)im * P.ldw_m;
        const int* idx_k = P.idx_k;
        const int64_t ldw_k = P.ldw_k;
#pragma unroll 8
        for (int k = kq; k < K; k += KSTEP) {
            const int ik = idx_k ? __ldg(idx_k + k) : k;
            const float v = live ? __ldg(wsrc + ik * ldw_k) : 0.f;
            Wd[k * MW + r] = v;
        }
    }

    // ---- output addressing: row m of this warp's slab goes to out0 (m < m_split) or out1
    const int mrow0 = m0 + wr * 16;
    const int o_rs = RS ? RS : a.p[pi].o_rs, m_split = a.p[pi].m_split;
    const bool slab_uniform = (mrow0 + 16 <= m_split) || (mrow0 >= m_split);
    const int slab_dst = (mrow0 >= m_split) ? 1 : 0;
    const int nrow_live = (M - mrow0 < 16) ? (M - mrow0) : 16;  // may be <= 0
    float* const ob = slab_dst ? a.p[pi].out1 + (int64_t)(mrow0 - m_split) * o_rs : a.p[pi].out0 + (int64_t)mrow0 * o_rs;
    const int64_t obs = slab_dst ? a.p[pi].o_bs1 : a.p[pi].o_bs0;
    __syncthreads();

    float2 acc[8][4];  // [row pair][column]
    int xoff[4];
    const uint32_t stage0 = smem_u32(stages), stage_bytes = (uint32_t)a.stage_floats * 4u, rs_bytes = (uint32_t)x_rs * 4u;
    const uint32_t w0 = smem_u32(Wd) + (uint32_t)wr * 64u;  // this warp's 16 rows

    int ti = rank, kc = 0, s = 0, prev_s = 0;
    uint32_t phase = 0, prev_phase = 0;
    int b0 = 0, ncol = 0, cbase = 0;
    for (int c = 0; c < nchunks; ++c) {
        // The slot of chunk c-1 is refilled with chunk c+NSTAGE-1 once every warp has released it.  Only warp 0
        // (the producer) waits for that; it is a consumer too, so the others have normally released the slot
        // before warp 0 itself gets here, and no warp ever waits for a CTA-wide barrier in steady state.
        if (warp == 0 && c > 0) mbar_wait(&empty[prev_s], prev_phase);
        produce();

        if (kc == 0) {
            int off0;
            tile_origin(ti, b0, off0);
            const int nb = (int)((a.batch - b0 < AB) ? (a.batch - b0) : AB);
            ncol = nb * J;
            if (WIN && ncol > off0 + CWT) ncol = off0 + CWT;  // the columns beyond belong to the next tile
            cbase = off0 + wc * 128 + lane;
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int tp = 0; tp < 4; ++tp) acc[r][tp] = make_float2(0.f, 0.f);
#pragma unroll
            for (int t = 0; t < 4; ++t) {
                const int cc = cbase + 32 * t;
                const int al = (J == 1) ? cc : (int)__umulhi((uint32_t)cc, jmagic);
                xoff[t] = (cc < ncol) ? 4 * (al * chunk_floats + j0 + (cc - al * J)) : 0;  // bytes
            }
        }
        mbar_wait(&full[s], phase);
        {
            // x address = (per-thread column offset) + (warp-uniform slot / row offset): the uniform part
            // stays on the uniform datapath, so the FMA pipe sees no address arithmetic
            const uint32_t ub = stage0 + (uint32_t)s * stage_bytes;
            const uint32_t wb = w0 + (uint32_t)(kc * KC) * (MW * 4);
            // RS: the four column addresses of this chunk; row kk is then an immediate offset kk * RS * 4
            uint32_t xb[4];
#pragma unroll
            for (int t = 0; t < 4; ++t) xb[t] = (uint32_t)xoff[t] + ub;
#pragma unroll 8
            for (int kk = 0; kk < KC; ++kk) {
                const uint32_t wa = wb + (uint32_t)kk * (MW * 4);
                const float4 wA = lds128(wa), wB = lds128(wa + 16), wC = lds128(wa + 32), wD = lds128(wa + 48);
                const uint32_t rowb = ub + (uint32_t)kk * rs_bytes;
                float2 x[4];
#pragma unroll
                for (int t = 0; t < 4; ++t) {
                    const float v = RS ? lds32(xb[t] + (uint32_t)kk * (uint32_t)(RS * 4)) : lds32(xoff[t] + rowb);
                    x[t] = make_float2(v, v);
                }
#pragma unroll
                for (int t = 0; t < 4; ++t) {
                    acc[0][t] = __ffma2_rn(make_float2(wA.x, wA.y), x[t], acc[0][t]);
                    acc[1][t] = __ffma2_rn(make_float2(wA.z, wA.w), x[t], acc[1][t]);
                    acc[2][t] = __ffma2_rn(make_float2(wB.x, wB.y), x[t], acc[2][t]);
                    acc[3][t] = __ffma2_rn(make_float2(wB.z, wB.w), x[t], acc[3][t]);
                    acc[4][t] = __ffma2_rn(make_float2(wC.x, wC.y), x[t], acc[4][t]);
                    acc[5][t] = __ffma2_rn(make_float2(wC.z, wC.w), x[t], acc[5][t]);
                    acc[6][t] = __ffma2_rn(make_float2(wD.x, wD.y), x[t], acc[6][t]);
                    acc[7][t] = __ffma2_rn(make_float2(wD.z, wD.w), x[t], acc[7][t]);
                }
            }
        }

        if (kc == NCH - 1 && nrow_live > 0) {
#pragma unroll
            for (int t = 0; t < 4; ++t) {
                const int cc = cbase + 32 * t;
                if (cc >= ncol) continue;
                const int al = (J == 1) ? cc : (int)__umulhi((uint32_t)cc, jmagic), j = cc - al * J;
                const int64_t b = (int64_t)b0 + al;
                if (slab_uniform && !ACC && nrow_live == 16) {
                    // the common case: a full slab of 16 rows, no predicates (with RS the row offsets are immediates)
                    float* dst = ob + b * obs + j;
                    if constexpr (RS > 0) {
#define CGTP_ST(r) stg_off<(r) * RS * 4>(dst, ((r) & 1) ? acc[(r) >> 1][t].y : acc[(r) >> 1][t].x);
                        CGTP_ST(0) CGTP_ST(1) CGTP_ST(2) CGTP_ST(3) CGTP_ST(4) CGTP_ST(5) CGTP_ST(6) CGTP_ST(7)
                        CGTP_ST(8) CGTP_ST(9) CGTP_ST(10) CGTP_ST(11) CGTP_ST(12) CGTP_ST(13) CGTP_ST(14) CGTP_ST(15)
#undef CGTP_ST
                    } else {
#pragma unroll
                        for (int r = 0; r < 16; ++r) dst[(int64_t)r * o_rs] = (r & 1) ? acc[r >> 1][t].y : acc[r >> 1][t].x;
                    }
                } else if (slab_uniform) {
                    float* dst = ob + b * obs + j;
                    float prev[16];
                    if (ACC) {
                        // all loads first: a load issued after a store to a possibly aliasing address would wait for it
#pragma unroll
                        for (int r = 0; r < 16; ++r) prev[r] = (r < nrow_live) ? __ldcg(dst + (int64_t)r * o_rs) : 0.f;
                    }
#pragma unroll
                    for (int r = 0; r < 16; ++r)
                        if (r < nrow_live) {
                            const float v = (r & 1) ? acc[r >> 1][t].y : acc[r >> 1][t].x;
                            dst[(int64_t)r * o_rs] = ACC ? prev[r] + v : v;
                        }
                } else {
#pragma unroll
                    for (int r = 0; r < 16; ++r) {
                        if (r >= nrow_live) continue;
                        const PfProblem& P = a.p[pi];
                        const int m = mrow0 + r;
                        float* dst = (m < m_split) ? P.out0 + b * P.o_bs0 + (int64_t)m * o_rs + j
                                                   : P.out1 + b * P.o_bs1 + (int64_t)(m - m_split) * o_rs + j;
                        const float v = (r & 1) ? acc[r >> 1][t].y : acc[r >> 1][t].x;
                        *dst = ACC ? *dst + v : v;
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive_cta(&empty[s]);
        prev_s = s;
        prev_phase = phase;
        if (++kc == NCH) { kc = 0; ti += cpr; }
        if (++s == NSTAGE) { s = 0; phase ^= 1u; }
    }
}

// ------------------------------------------------------------------------------------------------
// Host: configuration search and launch
// ------------------------------------------------------------------------------------------------

static inline bool al16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// Returns CGTP_OK and *handled = true if the fast kernel ran; *handled = false if the arguments do not
// meet its layout conditions (the caller then uses the generic kernel).
int launch_proj_fast(const ProjArgs* args, int nargs, Kind kind, cudaStream_t st, bool* handled)
{
    *handled = false;
    if (nargs < 1 || nargs > 2) return CGTP_OK;
    const int J = args[0].J;
    const int64_t batch = args[0].batch;
    int maxM = 0, maxK = 0;
    for (int i = 0; i < nargs; ++i) {
        const ProjArgs& g = args[i];
        if (g.J != J || g.batch != batch || g.x_rs != args[0].x_rs || g.accumulate != args[0].accumulate) return CGTP_OK;
        if (g.K < 2 || (g.K & 1) || g.M < 1 || g.x_rs < g.j0 + J || g.j0 < 0) return CGTP_OK;
        if (!al16(g.X) || (g.x_bs & 3)) return CGTP_OK;
        maxM = std::max(maxM, g.M);
        maxK = std::max(maxK, g.K);
    }
    if (batch <= 0 || J <= 0 || batch > 2000000000LL) return CGTP_OK;
    const int x_rs = args[0].x_rs;
    const bool wide = maxM <= 32;          // 32 rows x 512 columns, else 64 rows x 256 columns
    const int MW = wide ? 32 : 64, CWT = wide ? 512 : 256;
    const size_t wbytes = (size_t)maxK * MW * 4;
    const size_t budget = 226 * 1024;  // one CTA per SM
    if (wbytes + 2 * 4096 + 64 > budget) return CGTP_OK;

    // K chunk: divides every K, chunk bytes a multiple of 16
    int kcs[8], nkc = 0;
    for (int kc : {64, 32, 16, 8, 4, 2}) {
        bool ok = ((kc * x_rs) & 3) == 0;
        for (int i = 0; i < nargs; ++i) ok = ok && (args[i].K % kc == 0);
        if (ok) kcs[nkc++] = kc;
    }
    if (!nkc) return CGTP_OK;

    // search (AB, KC, NSTAGE): column efficiency first, then deep pipeline, then long chunks
    double best = -1.0;
    int bAB = 0, bKC = 0, bNS = 0;
    const int abmax = (int)std::min<int64_t>(batch, 64);
    for (int AB = 1; AB <= abmax; ++AB) {
        const int cols = AB * J;
        const int nsub = (cols + CWT - 1) / CWT;
        if (nsub > 4) break;
        const double eff = (double)cols / ((double)CWT * nsub);
        for (int i = 0; i < nkc; ++i) {
            const size_t sb = (size_t)AB * kcs[i] * x_rs * 4;
            for (int NS = 2; NS <= 3; ++NS) {
                if (64 + wbytes + NS * sb > budget) break;
                double score = eff;
                score *= (NS >= 3) ? 1.0 : 0.92;
                score *= (kcs[i] >= 64) ? 1.02 : (kcs[i] >= 16) ? 1.0 : (kcs[i] >= 8 ? 0.95 : 0.8);  // fewer chunk hand-overs
                score *= (nsub == 1) ? 1.0 : 0.97;  // sub-tiles re-read the stage from L2
                score -= 1e-4 * AB + 1e-5 * NS;      // ties: fewer atoms per stage, fewer stages
                if (score > best) { best = score; bAB = AB; bKC = kcs[i]; bNS = NS; }
            }
        }
    }
    if (best < 0.0) return CGTP_OK;
    const int slots_total = num_sms();

    // Window tiles: a tile is CWT consecutive flattened (atom, j) columns, so every tile is full and atoms straddle
    // tile boundaries; the stage then holds every atom the window touches (up to ABw).  Taken when it saves rounds of
    // the persistent CTAs after charging the extra staging traffic (boundary atoms are staged by two tiles).
    int window = 0;
    {
        const int ABw = (CWT + 2 * J - 2) / J;
        int wKC = 0, wNS = 0;
        for (int NS = 3; NS >= 2 && !wKC; --NS)
            for (int i = 0; i < nkc; ++i)
                if (kcs[i] >= 8 && 64 + wbytes + (size_t)NS * ABw * kcs[i] * x_rs * 4 <= budget) { wKC = kcs[i]; wNS = NS; break; }
        if (wKC && batch * (int64_t)J >= 4 * (int64_t)CWT) {
            const int nsub_g = (bAB * J + CWT - 1) / CWT;
            const int64_t tiles_g = (batch + bAB - 1) / bAB * nsub_g;
            const int64_t tiles_w = (batch * (int64_t)J + CWT - 1) / CWT;
            int nrb_tot = 0;
            for (int i = 0; i < nargs; ++i) nrb_tot += (args[i].M + MW - 1) / MW;
            const int per = std::max(1, slots_total / std::max(1, nrb_tot));
            // staging traffic per tile relative to the columns it computes: sub-tiles of a group re-stage the whole
            // group (factor nsub), a window stages the atoms it straddles (factor ABw J / CWT).  Measured (configs[3]):
            // the window pays off where it replaces sub-tiles (lmax = 16: 772 -> 588 us) and where it saves at least
            // ~6 % of the rounds at a factor <= 1.4 (configs[1]); elsewhere the extra staging costs more than it saves
            const double lf_g = nsub_g, lf_w = (double)ABw * J / CWT;
            const int64_t rounds_g = (tiles_g + per - 1) / per, rounds_w = (tiles_w + per - 1) / per;
            // sub-tiles of a group run on neighbouring CTAs at about the same time, so their re-staging is served by L2
            // as long as the CTAs do not drift apart; with operands of several times the L2 size it is not
            double xbytes = 0.0;
            for (int i = 0; i < nargs; ++i) xbytes += (double)batch * args[i].K * x_rs * 4.0;
            const bool beyond_l2 = xbytes > 4.0 * 126e6;
            if ((nsub_g > 1 && lf_w < lf_g && beyond_l2) || (lf_w <= 1.4 && 1.05 * rounds_w < (double)rounds_g)) {
                window = 1;
                bAB = ABw;
                bKC = wKC;
                bNS = wNS;
            }
        }
    }

    PfArgs a;
    a.nprob = nargs;
    a.J = J;
    a.batch = batch;
    a.AB = bAB;
    a.KC = bKC;
    a.NSTAGE = bNS;
    a.NSUB = window ? 1 : (bAB * J + CWT - 1) / CWT;
    a.stage_floats = bAB * bKC * x_rs;
    a.w_floats = maxK * MW;
    a.window = window;
    a.jmagic = (uint32_t)((1ull << 32) / (uint64_t)J) + 1u;
    const size_t smem = 64 + wbytes + (size_t)bNS * a.stage_floats * 4;
    const int ctas_per_sm = 1;
    const int slots = num_sms() * ctas_per_sm;

    // split the CTAs among (problem, row block) in proportion to their work (~ K per row block)
    int nrb[2] = {0, 0}, tot_rb = 0;
    double wsum = 0.0;
    for (int i = 0; i < nargs; ++i) {
        nrb[i] = (args[i].M + MW - 1) / MW;
        tot_rb += nrb[i];
        wsum += (double)nrb[i] * args[i].K;
    }
    const int64_t ntiles = window ? (batch * (int64_t)J + CWT - 1) / CWT : (batch + bAB - 1) / bAB * a.NSUB;
    if (ntiles * 64 > 2147483647LL) return CGTP_OK;  // 32-bit tile / chunk counters in the kernel
    a.ntiles = (int)ntiles;
    int begin = 0;
    for (int i = 0; i < nargs; ++i) {
        const ProjArgs& g = args[i];
        PfProblem& q = a.p[i];
        q.X = g.X; q.x_bs = g.x_bs; q.x_rs = g.x_rs; q.W = g.W; q.ldw_m = g.ldw_m; q.ldw_k = g.ldw_k;
        q.idx_m = g.idx_m; q.idx_k = g.idx_k; q.M = g.M; q.K = g.K; q.j0 = g.j0;
        q.out0 = g.out0; q.o_bs0 = g.o_bs0; q.out1 = g.out1; q.o_bs1 = g.o_bs1; q.m_split = g.m_split; q.o_rs = g.o_rs;
        q.nrb = nrb[i];
        int per = (int)((double)slots * g.K / wsum);
        if (per < 1) per = 1;
        if ((int64_t)per > ntiles) per = (int)ntiles;
        q.ctas_per_rb = per;
        q.cta_begin = begin;
        begin += per * nrb[i];
    }
    if (nargs == 1) a.p[1] = a.p[0];
    const int grid = begin;

    LaunchScope scope(kind, st);
    const bool acc = args[0].accumulate != 0;  // out += result (second pass of the parity-slot entry points)
    void (*kern)(PfArgs);
    if (window)
        kern = wide ? (acc ? proj_fast_kernel<2, 4, true, true> : proj_fast_kernel<2, 4, false, true>)
                    : (acc ? proj_fast_kernel<4, 2, true, true> : proj_fast_kernel<4, 2, false, true>);
    else
        kern = wide ? (acc ? proj_fast_kernel<2, 4, true, false> : proj_fast_kernel<2, 4, false, false>)
                    : (acc ? proj_fast_kernel<4, 2, true, false> : proj_fast_kernel<4, 2, false, false>);
    // compile-time row stride when X and every output share it ((lmax+1)^2 is odd for even lmax, so the odd strides of H
    // and T equal the dense ones: S1, S5 and M1 at the band limits of BASELINE.json's configs)
    bool same_rs = !acc;
    for (int i = 0; i < nargs; ++i) same_rs = same_rs && args[i].o_rs == x_rs;
    if (same_rs && !(kernel_path() & PATH_GENERIC_PROJ)) {
        switch (x_rs) {
#define CGTP_RS(V)                                                                                             \
    case V:                                                                                                    \
        kern = window ? (wide ? proj_fast_kernel<2, 4, false, true, V> : proj_fast_kernel<4, 2, false, true, V>)  \
                      : (wide ? proj_fast_kernel<2, 4, false, false, V> : proj_fast_kernel<4, 2, false, false, V>); \
        break;
            CGTP_RS(9) CGTP_RS(25) CGTP_RS(49) CGTP_RS(81) CGTP_RS(169) CGTP_RS(289) CGTP_RS(441)
#undef CGTP_RS
            default: break;
        }
    }
    CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CGTP_CUDA_CHECK(launch_pdl(kern, (unsigned)grid, (unsigned)kPfThreads, smem, st, a));
    CGTP_CUDA_CHECK(cudaGetLastError());
    *handled = true;
    return CGTP_OK;
}

}  // namespace cgtp
