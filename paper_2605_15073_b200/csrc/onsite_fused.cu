// onsite_fused.cu -- the whole on-site step S1-S5 (Eq.(35)-(41) PAPER.md:322-346, odd channels
// Eq.(11)-(12) :107-:111) in ONE persistent kernel: the projected coefficients H and the rank-space results T never leave
// the SM ("-> H on chip"), A and B are read once, `out` is written once.
//
// One CTA per SM, 16 warps = two independent warp groups (WG) of 8 warps.  A warp group owns a tile of NA atoms at a
// time and runs, with its own named barriers,
//   P  (S1)  H = W_a . A, W_b . B          lane = rank-channel pair, thread tile 2 channels x 13 coefficients, FFMA2 over the
//                                          pair; the coefficient rows come from the raw TMA-staged atom block through 16-byte
//                                          aligned 128-bit broadcast loads (the row misalignment k mod 4 is static under
//                                          4-fold unrolling), the weight pair from one 64-bit load;
//   core (S2a-S4b)                         the stage functions of onsite_core.cuh on groups of 16 columns; the group's warps
//                                          are split into an even and an odd sub-group that work concurrently on the
//                                          pointwise and the curl channels (own barriers, own F planes); T overwrites the
//                                          dead H rows in place;
//   Q  (S5)  out = W_out . T per sector    same mapping as P with lane = output-channel pair; the tile's `out` block is
//                                          staged in shared memory and leaves with one TMA bulk store.
// The two warp groups share the weights and the tables in shared memory and drift apart in phase, so the FMA-dense
// projection phases of one overlap the load/store-heavy transform phases of the other.  The next tile's A/B block is
// fetched by TMA during Q into the (dead) F planes.
//
// Taken when the tile fits shared memory (band limit <= 8, lmax_out <= lmax, N and C such that a tile of NA <= 8 atoms has
// whole groups); otherwise cgtp_onsite runs the four-launch path (proj_fast + onsite_core), which is also what
// CGTP_PATH_UNFUSED_ONSITE forces.  Summation orders: k ascending with one accumulator per output in P and Q (as
// proj_fast.cu); the core is the same code as onsite_core.cu.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <mutex>

#include "onsite_core.cuh"
#include "proj_tile.cuh"

namespace cgtp {

constexpr int kFusedThreads = 512;
constexpr int kWgWarps = 8;
constexpr int kFusedGW = 16;   // columns per core group

struct FusedTab {
    int ta_e, ta_o, wp, qf, qi, sched_e, sched_o, bytes;  // byte offsets into the table blob
    int UP2, UP4, QFS, QIS, SOFF, NQ;
    int maxi_e, maxi_o;
    int we, wo;  // warps of the even / odd sub-group (we + wo = 8)
};

struct FusedArgs {
    FusedTab tab;
    const void* blob;
    const float *A, *B;
    const float *W_a, *W_b, *W_out;
    const int *idx_in, *idx_out_e, *idx_out_o;
    int ldw_out;
    float* out;
    long long batch;
    int ntiles;
    int NA, N, C, Ce, Co;
    int lmax, lmax_out, L2, Lo2, L2s, U, Uh;
    int nsl_in, nsl_out;  // column tiles per row of P / Q
    // shared-memory byte offsets
    int off_blob, off_w, off_wg, wg_bytes;  // warp group w: off_wg + w * wg_bytes
    // inside a warp group's block: the A/B buffers (two when dbl: the next tile is fetched while this one is computed; else
    // one, overlaid by the F planes and refilled during Q), the staged `out` block, the F planes of the two sub-groups
    // (gc column groups each, so that gc groups share one barrier per stage), then Ha | Hb
    int off_ab0, off_ab1, off_ost, off_fe, off_fo, off_h;
    int dbl, gc;
};

__device__ __forceinline__ void bar_sync(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// S2a-S4b for the groups of one parity, run by the nsub warps of a sub-group (2 workers = half-warps per warp).
template <int LB, bool ODD>
__device__ __forceinline__ void core_groups(const FusedArgs& a, const CoreQParam<LB>& qp, const float* __restrict__ ta,
                                            const float* __restrict__ wp,
                                            const int* __restrict__ sched, int MAXI, float* __restrict__ F,
                                            float* __restrict__ Ha, const float* __restrict__ Hb, int col_base, int ngroups,
                                            int sub_warp, int nsub, int bar_id, int lane)
{
    constexpr int UB = core_uhmax(LB), RB = 2 * UB, GW = kFusedGW, MR = 2 * LB + 1;
    constexpr int plane = MR * RB * GW;
    const int col = lane & (GW - 1);
    const int worker = sub_warp * 2 + (lane >> 4), nworkers = nsub * 2;
    const int ne = a.Uh;
    const int eq = (a.U & 1) ? a.Uh - 1 : -1;  // odd U: the last northern node is the equator, its own mirror image
    constexpr int fgroup = (ODD ? 4 : 2) * plane;  // floats of one group's F planes
    for (int g0 = 0; g0 < ngroups; g0 += a.gc) {
        const int ng = (ngroups - g0 < a.gc) ? (ngroups - g0) : a.gc;
        // stage A: the worker -> item-list map rotates with the group, so that the ragged lists even out over a batch
        for (int gi = 0; gi < ng; ++gi) {
            const int c0 = col_base + (g0 + gi) * GW + col;
            const float* ha = Ha + (size_t)c0 * a.L2s;
            const float* hb = Hb + (size_t)c0 * a.L2s;
            float* Fg = F + (size_t)gi * fgroup;
            const int wk = (worker + gi) % nworkers;
            const int na = sched[0 * kMaxWorkers + wk];
            const int* ia = sched + 3 * kMaxWorkers + (0 * kMaxWorkers + wk) * MAXI;
            for (int k = 0; k < na; ++k) {
                if constexpr (!ODD) {
                    stage_a_even<LB, UB, GW>(ta, a.tab.UP4, ha, hb, Fg, Fg + plane, ia[k], a.lmax, 0, ne, col);
                } else {
                    const int m = ia[k] >> 1, f = ia[k] & 1;
                    stage_a_odd<LB, UB, GW>(ta, a.tab.UP2, f ? hb : ha, Fg + (2 * f) * plane, Fg + (2 * f + 1) * plane, m,
                                            a.lmax, 0, ne, col);
                }
            }
        }
        bar_sync(bar_id, nsub * 32);
        // stage B: (group, grid row) items dealt round-robin
        for (int it = worker; it < ng * RB; it += nworkers) {
            const int gi = it / RB, lr = it - gi * RB;
            const int e = (lr < UB) ? lr : lr - UB;
            if (e >= ne || (lr >= UB && e == eq)) continue;
            stage_b_p<LB, ODD, RB, GW>(qp, F + (size_t)gi * fgroup, plane, lr, a.tab.NQ, col);
        }
        bar_sync(bar_id, nsub * 32);
        // stage C: T overwrites the column's factor-1 row of H, dead since stage A
        for (int gi = 0; gi < ng; ++gi) {
            const int c0 = col_base + (g0 + gi) * GW + col;
            const int wk = (worker + gi) % nworkers;
            const int nc = sched[2 * kMaxWorkers + wk];
            const int* ic = sched + 3 * kMaxWorkers + (2 * kMaxWorkers + wk) * MAXI;
            for (int k = 0; k < nc; ++k)
                stage_c<LB, UB, GW>(wp, a.tab.UP4, F + (size_t)gi * fgroup, Ha + (size_t)c0 * a.L2s, ic[k], a.lmax_out, 0, ne, eq,
                                    true, col);
        }
        bar_sync(bar_id, nsub * 32);
    }
}

// P: thread item = (factor, atom, column tile sl, row tile ct); rows (rank channels, parity-sorted order) ct + nct * i.
__device__ __forceinline__ void phase_p(const FusedArgs& a, int wwarp, int lane, uint32_t sAB, uint32_t sW, float* Ha,
                                        float* Hb, int tile_floats)
{
    const int N = a.N, C = a.C, Ce = a.Ce, Co = a.Co, NA = a.NA, L2 = a.L2, L2s = a.L2s;
    const int nct = C / kTM, nsl = a.nsl_in;
    const int total = 2 * NA * nsl * nct;
    const bool mis = (L2 & 3) == 1;
    for (int q = wwarp * 32 + lane; q < total; q += kWgWarps * 32) {
        const int ct = q % nct;
        int r = q / nct;
        const int sl = r % nsl;
        r /= nsl;
        const int at = r % NA, f = r / NA;
        const int lm0 = sl * kTW;
        const int hi = (sl == nsl - 1) ? L2 : lm0 + kTW;
        float2 acc[2][kTJ];
#pragma unroll
        for (int p = 0; p < 2; ++p)
#pragma unroll
            for (int t = 0; t < kTJ; ++t) acc[p][t] = make_float2(0.f, 0.f);
        const uint32_t x0 = sAB + (uint32_t)(f * tile_floats + at * N * L2 + lm0) * 4u;
        const uint32_t w0 = sW + (uint32_t)(f * N * C + ct * kTM) * 4u;
        if (mis) proj_tile<true>(acc, x0, (uint32_t)L2 * 4u, w0, (uint32_t)C * 4u, N);
        else proj_tile<false>(acc, x0, (uint32_t)L2 * 4u, w0, (uint32_t)C * 4u, N);
        float* Hf = f ? Hb : Ha;
#pragma unroll
        for (int i = 0; i < kTM; ++i) {
            const int c = ct + nct * i;
            float* d = Hf + (size_t)((c < Ce) ? at * Ce + c : NA * Ce + at * Co + (c - Ce)) * L2s + lm0;
#pragma unroll
            for (int t = 0; t < kTJ; ++t)
                if (lm0 + t < hi) d[t] = (i & 1) ? acc[i >> 1][t].y : acc[i >> 1][t].x;
        }
    }
}

// Q: thread item = (sector, atom, column tile, row tile); rows = output channels jt + nnt * i; the T rows sit in place of
// the factor-1 rows of H (stride L2s, 1 mod 4).
__device__ __forceinline__ void phase_q(const FusedArgs& a, int wwarp, int lane, uint32_t sHa, uint32_t sW, float* OST)
{
    const int N = a.N, C = a.C, Ce = a.Ce, Co = a.Co, NA = a.NA, Lo2 = a.Lo2, L2s = a.L2s;
    const int nnt = N / kTM, nsl = a.nsl_out;
    const int total = 2 * NA * nsl * nnt;
    for (int q = wwarp * 32 + lane; q < total; q += kWgWarps * 32) {
        const int jt = q % nnt;
        int r = q / nnt;
        const int sl = r % nsl;
        r /= nsl;
        const int at = r % NA, s = r / NA;
        const int lm0 = sl * kTW;
        const int hi = (sl == nsl - 1) ? Lo2 : lm0 + kTW;
        const int Cs = s ? Co : Ce;
        float2 acc[2][kTJ];
#pragma unroll
        for (int p = 0; p < 2; ++p)
#pragma unroll
            for (int t = 0; t < kTJ; ++t) acc[p][t] = make_float2(0.f, 0.f);
        const uint32_t x0 = sHa + (uint32_t)(((s ? NA * Ce : 0) + at * Cs) * L2s + lm0) * 4u;
        const uint32_t w0 = sW + (uint32_t)(2 * N * C + (s ? Ce * N : 0) + jt * kTM) * 4u;
        proj_tile<true>(acc, x0, (uint32_t)L2s * 4u, w0, (uint32_t)N * 4u, Cs);
#pragma unroll
        for (int i = 0; i < kTM; ++i) {
            float* d = OST + (size_t)((at * 2 + s) * N + jt + nnt * i) * Lo2 + lm0;
#pragma unroll
            for (int t = 0; t < kTJ; ++t)
                if (lm0 + t < hi) d[t] = (i & 1) ? acc[i >> 1][t].y : acc[i >> 1][t].x;
        }
    }
}

template <int LB>
__global__ void __launch_bounds__(kFusedThreads, 1) onsite_fused_kernel(const __grid_constant__ FusedArgs a,
                                                                        const __grid_constant__ CoreQParam<LB> qp)
{
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* bar_tab = reinterpret_cast<uint64_t*>(smem);
    uint64_t* bar_ab = reinterpret_cast<uint64_t*>(smem + 16);  // [2 warp groups][2 buffers]
    const unsigned char* blob = smem + a.off_blob;
    float* Wsm = reinterpret_cast<float*>(smem + a.off_w);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wg = warp / kWgWarps, wwarp = warp % kWgWarps, wtid = tid - wg * (kWgWarps * 32);
    const int N = a.N, C = a.C, Ce = a.Ce, Co = a.Co, NA = a.NA, L2 = a.L2, Lo2 = a.Lo2, L2s = a.L2s;

    if (tid == 0) {
        mbar_init(bar_tab, 1);
        for (int i = 0; i < 4; ++i) mbar_init(&bar_ab[i], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) {
        mbar_arrive_expect_tx(bar_tab, (uint32_t)a.tab.bytes);
        tma_load_span(smem + a.off_blob, a.blob, (uint32_t)a.tab.bytes, bar_tab);
    }

    // this warp group's shared memory
    unsigned char* wgm = smem + a.off_wg + (size_t)wg * a.wg_bytes;
    float* ABuf[2] = {reinterpret_cast<float*>(wgm + a.off_ab0), reinterpret_cast<float*>(wgm + a.off_ab1)};
    float* OST = reinterpret_cast<float*>(wgm + a.off_ost);
    float* Ha = reinterpret_cast<float*>(wgm + a.off_h);
    const int ncol = NA * C;
    float* Hb = Ha + (size_t)ncol * L2s;
    const int tile_floats = NA * N * L2;  // one factor

    auto load_tile = [&](int tile, int buf) {  // one thread of the warp group
        const long long b0 = (long long)tile * NA;
        const int nb = (int)((a.batch - b0 < NA) ? (a.batch - b0) : NA);
        const uint32_t bytes = (uint32_t)nb * N * L2 * 4u;
        uint64_t* bar = &bar_ab[wg * 2 + buf];
        mbar_arrive_expect_tx(bar, 2 * bytes);
        tma_load_span(ABuf[buf], a.A + b0 * N * L2, bytes, bar);
        tma_load_span(ABuf[buf] + tile_floats, a.B + b0 * N * L2, bytes, bar);
    };
    int tile = blockIdx.x * 2 + wg;
    const int tile_step = gridDim.x * 2;
    if (wtid == 0 && tile < a.ntiles) load_tile(tile, 0);

    // ---- weights -> shared memory in the order the projection tiles read them: Wp[k][tile][i], the 8 output rows of a
    // tile being tile + ntiles * i (rows of one thread 8 * stride apart: conflict-free stores of the results)
    {
        const int nct = C / kTM, nnt = N / kTM;
        float* Wa_p = Wsm;
        float* Wb_p = Wsm + (size_t)N * C;
        for (int t = tid; t < N * C; t += kFusedThreads) {
            const int c = t / N, k = t - c * N;
            const int row = a.idx_in ? __ldg(a.idx_in + c) : c;
            const int d = (k * nct + c % nct) * kTM + c / nct;
            Wa_p[d] = __ldg(a.W_a + (size_t)row * N + k);
            Wb_p[d] = __ldg(a.W_b + (size_t)row * N + k);
        }
        float* Wo = Wsm + (size_t)2 * N * C;
        for (int s = 0; s < 2; ++s) {
            const int Cs = s ? Co : Ce;
            const int* idx = s ? a.idx_out_o : a.idx_out_e;
            float* Wo_s = Wo + (s ? (size_t)Ce * N : 0);
            for (int t = tid; t < N * Cs; t += kFusedThreads) {
                const int n = t / Cs, k = t - n * Cs;
                const int cidx = idx ? __ldg(idx + k) : (s ? Ce + k : k);
                Wo_s[(k * nnt + n % nnt) * kTM + n / nnt] = __ldg(a.W_out + (size_t)n * a.ldw_out + cidx);
            }
        }
    }
    mbar_wait(bar_tab, 0);
    __syncthreads();

    const float* ta_e = reinterpret_cast<const float*>(blob + a.tab.ta_e);
    const float* ta_o = reinterpret_cast<const float*>(blob + a.tab.ta_o);
    const float* wp = reinterpret_cast<const float*>(blob + a.tab.wp);
    const int* sched_e = reinterpret_cast<const int*>(blob + a.tab.sched_e);
    const int* sched_o = reinterpret_cast<const int*>(blob + a.tab.sched_o);

    const int bar_full = 1 + 3 * wg, bar_e = 2 + 3 * wg, bar_o = 3 + 3 * wg;
    const uint32_t sHa = smem_u32(Ha), sW = smem_u32(Wsm);

    uint32_t phases = 0;  // bit b: parity to wait for on buffer b
    int buf = 0;
    for (; tile < a.ntiles; tile += tile_step) {
        const long long b0 = (long long)tile * NA;
        const int nb = (int)((a.batch - b0 < NA) ? (a.batch - b0) : NA);
        // two buffers: the other one was released by the barrier after the previous tile's P
        if (a.dbl && wtid == 0 && tile + tile_step < a.ntiles) load_tile(tile + tile_step, buf ^ 1);
        mbar_wait(&bar_ab[wg * 2 + buf], (phases >> buf) & 1u);
        phases ^= 1u << buf;
        const uint32_t sAB = smem_u32(ABuf[buf]);

        // ---- P (S1, Eq.(35)): H_f[col][lm] = sum_n W_f[c][n] X_f[a][n][lm]
        phase_p(a, wwarp, lane, sAB, sW, Ha, Hb, tile_floats);
        // the previous tile's bulk store must have read OST before the F planes (which overlay it) are rewritten
        if (wtid == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        bar_sync(bar_full, kWgWarps * 32);

        // ---- core (S2a-S4b): even and odd sub-groups side by side
        if (wwarp < a.tab.we) {
            if (Ce > 0)
                core_groups<LB, false>(a, qp, ta_e, wp, sched_e, a.tab.maxi_e, reinterpret_cast<float*>(wgm + a.off_fe), Ha,
                                       Hb, 0, NA * Ce / kFusedGW, wwarp, a.tab.we, bar_e, lane);
        } else {
            if (Co > 0)
                core_groups<LB, true>(a, qp, ta_o, wp, sched_o, a.tab.maxi_o,
                                      reinterpret_cast<float*>(wgm + a.off_fo), Ha, Hb, NA * Ce, NA * Co / kFusedGW,
                                      wwarp - a.tab.we, a.tab.wo, bar_o, lane);
        }
        fence_async_smem();  // generic writes to the F planes before the async-proxy write of the next A/B block
        bar_sync(bar_full, kWgWarps * 32);
        if (!a.dbl && wtid == 0 && tile + tile_step < a.ntiles) load_tile(tile + tile_step, 0);

        // ---- Q (S5, Eq.(41)): out[a][s][n][lm] = sum_{k in sector s} W_out[n][c_k] T[col(a,k)][lm]
        phase_q(a, wwarp, lane, sHa, sW, OST);
        fence_async_smem();
        bar_sync(bar_full, kWgWarps * 32);
        if (wtid == 0) {
            tma_store_1d(a.out + b0 * 2 * N * Lo2, OST, (uint32_t)nb * 2u * N * Lo2 * 4u);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
        if (a.dbl) buf ^= 1;
    }
    if (wtid == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// ------------------------------------------------------------------------------------------------
// Host: table blob (both parities' stage-A tables, shared analysis / azimuthal tables, one schedule per sub-group)
// ------------------------------------------------------------------------------------------------
struct FusedPlan {
    int dev, lmax, lmax_out, we, wo;
    FusedTab tab;
    const void* blob;
    std::vector<float> QF, QI;  // host copies of the azimuthal tables: passed to the kernel as a parameter (CoreQParam)
};
static std::mutex g_fused_mu;
static std::vector<FusedPlan*> g_fused_plans;

static const FusedPlan* get_fused_plan(const Plan* p, int we, int wo)
{
    std::lock_guard<std::mutex> lk(g_fused_mu);
    for (FusedPlan* f : g_fused_plans)
        if (f->dev == p->dev && f->lmax == p->lmax && f->lmax_out == p->lmax_out && f->we == we && f->wo == wo) return f;

    FusedTab t;
    std::memset(&t, 0, sizeof t);
    CoreTab ce, co;
    std::memset(&ce, 0, sizeof ce);
    std::memset(&co, 0, sizeof co);
    std::vector<float> TAe, TAo, WP, WP2, QF, QF2, QI, QI2;
    core_host_tables(p, false, ce, TAe, WP, QF, QI);
    core_host_tables(p, true, co, TAo, WP2, QF2, QI2);
    t.UP2 = co.UP2; t.UP4 = ce.UP4; t.QFS = ce.QFS; t.QIS = ce.QIS; t.SOFF = ce.SOFF; t.NQ = ce.NQ;
    t.we = we; t.wo = wo;

    auto make_sched = [&](bool odd, int nwarps, int* maxi_out) {
        std::vector<std::pair<int, int>> items[3];
        stage_items(p, odd, items);
        const int nworkers = std::max(1, 2 * nwarps);
        std::vector<std::vector<int>> asg[3];
        int maxi = 1;
        for (int s = 0; s < 3; ++s) {
            int mk;
            lpt_assign(items[s], nworkers, asg[s], &mk);
            for (auto& v : asg[s]) maxi = std::max(maxi, (int)v.size());
        }
        std::vector<int> sched((size_t)3 * kMaxWorkers + (size_t)3 * kMaxWorkers * maxi, 0);
        for (int s = 0; s < 3; ++s)
            for (int wi = 0; wi < nworkers; ++wi) {
                sched[s * kMaxWorkers + wi] = (int)asg[s][wi].size();
                for (size_t k = 0; k < asg[s][wi].size(); ++k)
                    sched[3 * kMaxWorkers + ((size_t)s * kMaxWorkers + wi) * maxi + k] = asg[s][wi][k];
            }
        *maxi_out = maxi;
        return sched;
    };
    std::vector<int> se = make_sched(false, we, &t.maxi_e), so = make_sched(true, wo, &t.maxi_o);

    std::vector<unsigned char> blob;
    auto append = [&](const void* src, size_t bytes) {
        const size_t off = blob.size();
        blob.resize(off + (bytes + 15) / 16 * 16);
        std::memcpy(blob.data() + off, src, bytes);
        return (int)off;
    };
    t.ta_e = append(TAe.data(), TAe.size() * 4);
    t.ta_o = append(TAo.data(), TAo.size() * 4);
    t.wp = append(WP.data(), WP.size() * 4);
    t.qf = append(QF.data(), QF.size() * 4);
    t.qi = append(QI.data(), QI.size() * 4);
    t.sched_e = append(se.data(), se.size() * 4);
    t.sched_o = append(so.data(), so.size() * 4);
    t.bytes = (int)blob.size();

    void* d = nullptr;
    if (cudaMalloc(&d, blob.size()) != cudaSuccess ||
        cudaMemcpy(d, blob.data(), blob.size(), cudaMemcpyHostToDevice) != cudaSuccess) {
        set_error("onsite fused plan: device upload failed: %s", cudaGetErrorString(cudaGetLastError()));
        return nullptr;
    }
    FusedPlan* f = new FusedPlan;
    f->dev = p->dev; f->lmax = p->lmax; f->lmax_out = p->lmax_out; f->we = we; f->wo = wo;
    f->tab = t;
    f->blob = d;
    f->QF = QF;
    f->QI = QI;
    g_fused_plans.push_back(f);
    return f;
}

static inline int al128(int x) { return (x + 127) / 128 * 128; }
template <int LB>
static int launch_fused_t(const FusedArgs& a, const FusedPlan* fp, int smem, int64_t grid, cudaStream_t st)
{
    CoreQParam<LB> qp;
    std::memset(&qp, 0, sizeof qp);
    std::memcpy(qp.qf, fp->QF.data(), std::min(sizeof qp.qf, fp->QF.size() * sizeof(float)));
    std::memcpy(qp.qi, fp->QI.data(), std::min(sizeof qp.qi, fp->QI.size() * sizeof(float)));
    auto kern = onsite_fused_kernel<LB>;
    CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    LaunchScope scope(K_ONSITE_FUSED, st);
    kern<<<(unsigned)grid, kFusedThreads, smem, st>>>(a, qp);
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

int launch_onsite_fused(const Plan* p, int N, int C, int Ce, int Co, const float* A, const float* B, const float* W_a,
                        const float* W_b, const int* idx_in, const float* W_out, int ldw_out, const int* idx_out_e,
                        const int* idx_out_o, float* out, int64_t batch, cudaStream_t st, bool* handled)
{
    *handled = false;
    const int LB = p->LB;
    if (LB > 8 || p->lmax_out > p->lmax || N % kTM != 0 || C % kTM != 0 || Ce % 4 != 0 || Co % 4 != 0 || batch <= 0)
        return CGTP_OK;
    // Taken where it was measured faster than the four launches (B200, DESIGN.md 5.11 / 5.14): narrow projections
    // (N C <= 256) at band limits >= 4 (N = C = 16, 20000 atoms, lmax 4 / 5 / 6: 160 / 206 / 298 vs 195 / 269 / 389 us) and
    // problems so small that launch latency dominates (configs[0]: 23 vs 38 us).  Elsewhere the four launches win: the
    // small band limits have the register core of onsite_reg.cu and the projections of proj_fast.cu address with
    // compile-time strides (configs[1]: 243 us in four launches, 257 us here; N = C = 32, configs[3], lmax 2 / 4: 78 / 175 vs
    // 116 / 261 us).  CGTP_PATH_FUSED_ONSITE forces the kernel for every shape it supports (tests, bench).
    // (N = C = 8, 30000 atoms, lmax 2: 83 vs 123 us; N = C = 64, lmax 6, 256 atoms: 32 vs 48 us, 1024 atoms: 85 vs 83 us)
    const bool narrow = (int64_t)N * C <= 64 || ((int64_t)N * C <= 256 && LB >= 4);
    const bool tiny = batch * (int64_t)C * p->L2 <= (1 << 17) || batch <= 512;
    if (!narrow && !tiny && !(kernel_path() & PATH_FUSED_ONSITE)) return CGTP_OK;
    // warps of the two sub-groups by estimated work: a curl group costs about 1.9 pointwise groups (configs[1]: 3 + 5 warps 260 us, 4 + 4 warps 304 us -- ten grid rows on ten half-warp workers is one round of stage B)
    int we = 8, wo = 0;
    if (Ce == 0) { we = 0; wo = 8; }
    else if (Co > 0) {
        const double ce = (double)Ce, co = 1.9 * Co;
        we = (int)std::lround(8.0 * ce / (ce + co));
        we = std::min(7, std::max(1, we));
        wo = 8 - we;
    }
    const int MR = 2 * LB + 1, RB = 2 * core_uhmax(LB);
    const FusedPlan* fp = get_fused_plan(p, we, wo);
    if (!fp) return CGTP_ERR_CUDA;
    FusedArgs a;
    std::memset(&a, 0, sizeof a);
    a.N = N; a.C = C; a.Ce = Ce; a.Co = Co;
    a.lmax = p->lmax; a.lmax_out = p->lmax_out; a.L2 = p->L2; a.Lo2 = p->Lo2; a.L2s = p->L2 | 1; a.U = p->U; a.Uh = p->Uh;
    a.nsl_in = proj_num_slices(p->L2);
    a.nsl_out = proj_num_slices(p->Lo2);
    a.tab = fp->tab;
    a.blob = fp->blob;
    a.off_blob = 64;
    a.off_w = al128(a.off_blob + fp->tab.bytes);
    a.off_wg = al128(a.off_w + 3 * N * C * 4);
    const int fe_bytes = (Ce > 0 ? 2 : 0) * MR * RB * kFusedGW * 4, fo_bytes = (Co > 0 ? 4 : 0) * MR * RB * kFusedGW * 4;
    // Atoms per tile NA (whole column groups), concurrent groups gc and buffering: a roomy layout (two A/B buffers, the F
    // planes of gc groups next to them) when shared memory holds it -- more atoms per tile and fewer barriers amortise the
    // per-tile latencies of small shapes --, else the tight layout (one A/B buffer under the F planes, one group at a time).
    int NA = 0, smem = 0;
    auto plan = [&](int na, bool dbl, int gc) -> int {
        const int ab_bytes = al128(2 * na * N * p->L2 * 4 + 64), ost_bytes = al128(na * 2 * N * p->Lo2 * 4);
        const int f_bytes = al128(gc * fe_bytes) + al128(gc * fo_bytes);
        int off = 0, off_ab0, off_ab1, off_ost, off_f;
        if (dbl) {
            off_ab0 = 0; off_ab1 = ab_bytes; off = 2 * ab_bytes;
            off_ost = off; off_f = off; off += std::max(ost_bytes, f_bytes);  // `out` staging under the F planes
        } else {
            off_ab0 = off_ab1 = 0; off_ost = ab_bytes; off_f = 0;
            off = std::max(ab_bytes + ost_bytes, f_bytes);
        }
        const int off_h = al128(off);
        const int wg_bytes = al128(off_h + 2 * na * C * a.L2s * 4 + 64);
        const int total = a.off_wg + 2 * wg_bytes;
        if (total > 227 * 1024) return 0;
        a.off_ab0 = off_ab0; a.off_ab1 = off_ab1; a.off_ost = off_ost; a.off_fe = off_f; a.off_fo = off_f + al128(gc * fe_bytes);
        a.off_h = off_h; a.wg_bytes = wg_bytes; a.dbl = dbl ? 1 : 0; a.gc = gc;
        return total;
    };
    for (int na = 8; na >= 1 && !NA; na /= 2) {
        if ((na * Ce) % kFusedGW != 0 || (na * Co) % kFusedGW != 0) continue;
        if (na > 1 && (batch + na - 1) / na < (int64_t)8 * num_sms()) continue;  // keep a few tiles per warp group
        const int ng = std::max(na * Ce, na * Co) / kFusedGW;
        for (int gc = std::min(ng, 8); gc >= 1 && !NA; gc /= 2)
            if ((smem = plan(na, true, gc)) != 0) NA = na;
    }
    for (int na = 1; na <= 8 && !NA; na *= 2) {
        if ((na * Ce) % kFusedGW != 0 || (na * Co) % kFusedGW != 0) continue;
        if ((smem = plan(na, false, 1)) != 0) NA = na;
        break;
    }
    if (!NA) return CGTP_OK;  // the four-launch path takes it
    a.NA = NA;
    *handled = true;
    a.A = A; a.B = B; a.W_a = W_a; a.W_b = W_b; a.W_out = W_out;
    a.idx_in = idx_in; a.idx_out_e = idx_out_e; a.idx_out_o = idx_out_o; a.ldw_out = ldw_out;
    a.out = out;
    a.batch = batch;
    const int64_t ntiles = (batch + NA - 1) / NA;
    if (ntiles > 2147483647LL / 4) { set_error("onsite fused: batch too large"); return CGTP_ERR_UNSUPPORTED; }
    a.ntiles = (int)ntiles;
    int64_t grid = std::min<int64_t>(num_sms(), (ntiles + 1) / 2);
    switch (LB) {
#define CGTP_CASE(Bn) \
    case Bn:          \
        return launch_fused_t<Bn>(a, fp, smem, grid, st);
        CGTP_CASE(1) CGTP_CASE(2) CGTP_CASE(3) CGTP_CASE(4) CGTP_CASE(5) CGTP_CASE(6) CGTP_CASE(8)
#undef CGTP_CASE
    }
    *handled = false;
    return CGTP_OK;
}

}  // namespace cgtp
