// proj_multi.cu -- the channel projections with l-dependent CP weights (c_{cnl} of Eq.(35) PAPER.md:322 and Eq.(47)
// :398, lambda_c^{(nl)} of Eq.(41) :346 and Eq.(55) :427) as ONE launch over all degrees: the streaming kernel
// of proj_fast.cu (same staging ring, same packed-FMA main loop, same summation order) with a table of problems, one per
// (degree l, factor): the problem fixes the weight matrix W[l], the column range l^2 .. l^2 + 2l of the feature rows and
// its own number of atoms per tile, and owns a share of the persistent CTAs in proportion to its work.  A launch per
// degree gave every CTA one to three tiles (30 us per launch whatever the degree: prologue-bound).
#include <algorithm>

#include "sht.cuh"

namespace cgtp {

constexpr int kPfThreads = 256;
constexpr int kPmMaxProblems = 44;  // 2 factors x 22 degrees

struct PmProblem {
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
    int J;         // used columns per atom (2l+1)
    int AB;        // atoms per tile
    int ntiles;    // tiles per row block
    uint32_t jmagic;
    int nrb;       // row blocks of this problem
    int cta_begin; // first CTA (blockIdx.x) serving this problem
    int ctas_per_rb;
};

struct PmArgs {
    PmProblem p[kPmMaxProblems];
    int nprob;
    int64_t batch;
    int KC, NSTAGE;
    int stage_floats;  // max over the problems of AB * KC * x_rs
    int w_floats;      // Kmax * MW
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

__device__ __forceinline__ void mbar_arrive_cta(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

template <int RW, int CWP>
__global__ void __launch_bounds__(kPfThreads, 1) proj_multi_kernel(const __grid_constant__ PmArgs a)
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

    constexpr bool ACC = false, WIN = false;
    // which (problem, row block, rank within the row block) this CTA serves: problems are (degree, factor) pairs with
    // their own column count, atoms per tile and weights; the fields are copied to registers once
    int pi = 0;
    while (pi + 1 < a.nprob && (int)blockIdx.x >= a.p[pi + 1].cta_begin) ++pi;
    const PmProblem& P0 = a.p[pi];
    const float* const X = P0.X;
    const int64_t x_bs = P0.x_bs;
    const int x_rs = P0.x_rs;
    const int M = P0.M;
    const int K = P0.K;
    const int cpr = P0.ctas_per_rb;
    const int j0 = P0.j0;
    const int local = blockIdx.x - P0.cta_begin;
    const int rb = local / cpr, rank = local - rb * cpr;
    const int m0 = rb * MW;
    const int J = P0.J, AB = P0.AB, NSUB = 1, NSTAGE = a.NSTAGE, KC = a.KC;
    const uint32_t jmagic = P0.jmagic;  // cc / J == umulhi(cc, jmagic) for cc < 2^16

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
    const int ntiles = P0.ntiles;
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
    // programmatic dependent launch (common.cuh): everything read below is a caller input or a predecessor's output
    pdl_launch_dependents();
    pdl_wait();
    for (int i = 0; i < NSTAGE - 1; ++i) produce();

    // ---- weights: Wd[k][r] = W[idx_m[m0+r]][idx_k[k]].  Thread = fixed row r,
    // strided k: the loads of different k are independent and stay in flight together.
    {
        const PmProblem& P = a.p[pi];
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
    const int o_rs = a.p[pi].o_rs, m_split = a.p[pi].m_split;
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
#pragma unroll 8
            for (int kk = 0; kk < KC; ++kk) {
                const uint32_t wa = wb + (uint32_t)kk * (MW * 4);
                const float4 wA = lds128(wa), wB = lds128(wa + 16), wC = lds128(wa + 32), wD = lds128(wa + 48);
                const uint32_t rowb = ub + (uint32_t)kk * rs_bytes;
                float2 x[4];
#pragma unroll
                for (int t = 0; t < 4; ++t) {
                    const float v = lds32(xoff[t] + rowb);
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
                if (slab_uniform) {
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
                        const PmProblem& P = a.p[pi];
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
// Host
// ------------------------------------------------------------------------------------------------

static inline bool pm_al16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// One launch for up to kPmMaxProblems projection problems that share batch, K and the row stride of X but differ in
// their column range (j0, J) and weights.  *handled = false when the layout conditions do not hold (the caller then
// launches the problems one by one through launch_proj).
int launch_proj_multi(const ProjArgs* args, int nargs, Kind kind, cudaStream_t st, bool* handled)
{
    *handled = false;
    if (nargs < 1 || nargs > kPmMaxProblems) return CGTP_OK;
    const int64_t batch = args[0].batch;
    const int K = args[0].K, x_rs = args[0].x_rs;
    int maxM = 0;
    for (int i = 0; i < nargs; ++i) {
        const ProjArgs& g = args[i];
        if (g.batch != batch || g.K != K || g.x_rs != x_rs || g.accumulate) return CGTP_OK;
        if (g.J < 1 || g.j0 < 0 || g.j0 + g.J > x_rs || g.M < 1) return CGTP_OK;
        if (!pm_al16(g.X) || (g.x_bs & 3)) return CGTP_OK;
        maxM = std::max(maxM, g.M);
    }
    if (K < 2 || (K & 1) || batch <= 0 || batch > 2000000000LL) return CGTP_OK;
    const bool wide = maxM <= 32;  // 32 rows x 512 columns, else 64 rows x 256 columns
    const int MW = wide ? 32 : 64, CWT = wide ? 512 : 256;
    const size_t wbytes = (size_t)K * MW * 4;
    const size_t budget = 226 * 1024;
    if (wbytes + 2 * 4096 + 64 > budget) return CGTP_OK;

    // (KC, NSTAGE): fewest tile-steps sum_i tiles_i * K over the problems; the atoms per tile of a problem are bounded
    // by the tile width and by the stage size (whole feature rows are staged)
    double best = 1e300;
    int bKC = 0, bNS = 0;
    for (int kc : {64, 32, 16, 8, 4}) {
        if (K % kc || ((kc * x_rs) & 3)) continue;
        for (int NS = 3; NS >= 2; --NS) {
            const size_t sb = (budget - 64 - wbytes) / NS / 16 * 16;
            const int abcap = (int)(sb / ((size_t)kc * x_rs * 4));
            if (abcap < 1) continue;
            double tiles = 0.0;
            for (int i = 0; i < nargs; ++i) {
                int AB = std::min<int64_t>(std::min(CWT / args[i].J, abcap), batch);
                if (AB < 1) AB = 1;
                tiles += (double)((batch + AB - 1) / AB) * ((args[i].M + MW - 1) / MW);
            }
            // short chunks pay a ring hand-over every kc steps of the contraction (measured at configs[1]: S1 0.198 ms
            // with kc = 16, 0.220 with 32, 0.324 with 8, 0.656 with 4 although the tile count falls with kc)
            double cost = tiles * (NS >= 3 ? 1.0 : 1.08) * (kc >= 16 ? 1.0 : kc >= 8 ? 1.7 : 3.5);
            if (cost < best) { best = cost; bKC = kc; bNS = NS; }
        }
    }
    if (!bKC) return CGTP_OK;
    const size_t sb = (budget - 64 - wbytes) / bNS / 16 * 16;
    const int abcap = (int)(sb / ((size_t)bKC * x_rs * 4));

    PmArgs a;
    a.nprob = nargs;
    a.batch = batch;
    a.KC = bKC;
    a.NSTAGE = bNS;
    a.w_floats = K * MW;
    int maxAB = 1;
    double wsum = 0.0;
    int64_t tiles_i[kPmMaxProblems];
    for (int i = 0; i < nargs; ++i) {
        const ProjArgs& g = args[i];
        PmProblem& q = a.p[i];
        int AB = (int)std::min<int64_t>(std::min(CWT / g.J, abcap), batch);
        if (AB < 1) AB = 1;
        if (AB * g.J > CWT) return CGTP_OK;  // J wider than a tile: not a per-degree problem
        maxAB = std::max(maxAB, AB);
        q.X = g.X; q.x_bs = g.x_bs; q.x_rs = g.x_rs; q.W = g.W; q.ldw_m = g.ldw_m; q.ldw_k = g.ldw_k;
        q.idx_m = g.idx_m; q.idx_k = g.idx_k; q.M = g.M; q.K = g.K;
        q.out0 = g.out0; q.o_bs0 = g.o_bs0; q.out1 = g.out1; q.o_bs1 = g.o_bs1; q.m_split = g.m_split; q.o_rs = g.o_rs;
        q.j0 = g.j0; q.J = g.J; q.AB = AB;
        tiles_i[i] = (batch + AB - 1) / AB;
        if (tiles_i[i] * 64 > 2147483647LL) return CGTP_OK;
        q.ntiles = (int)tiles_i[i];
        q.jmagic = (uint32_t)((1ull << 32) / (uint64_t)g.J) + 1u;
        q.nrb = (g.M + MW - 1) / MW;
        wsum += (double)q.nrb * (double)tiles_i[i];
    }
    a.stage_floats = maxAB * bKC * x_rs;
    const size_t smem = 64 + wbytes + (size_t)bNS * a.stage_floats * 4;
    if (smem > budget) return CGTP_OK;
    const int slots = num_sms();
    int begin = 0;
    for (int i = 0; i < nargs; ++i) {
        PmProblem& q = a.p[i];
        int per = (int)((double)slots * (double)tiles_i[i] / wsum);
        if (per < 1) per = 1;
        if ((int64_t)per > tiles_i[i]) per = (int)tiles_i[i];
        q.ctas_per_rb = per;
        q.cta_begin = begin;
        begin += per * q.nrb;
    }
    for (int i = nargs; i < kPmMaxProblems; ++i) a.p[i] = a.p[0];
    const int grid = begin;

    LaunchScope scope(kind, st);
    void (*kern)(const PmArgs) = wide ? proj_multi_kernel<2, 4> : proj_multi_kernel<4, 2>;
    CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CGTP_CUDA_CHECK(launch_pdl(kern, (unsigned)grid, (unsigned)kPfThreads, smem, st, a));
    CGTP_CUDA_CHECK(cudaGetLastError());
    *handled = true;
    return CGTP_OK;
}

}  // namespace cgtp
