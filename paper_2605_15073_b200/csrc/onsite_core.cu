// onsite_core.cu -- fast fused on-site core (rows S2a, S2b, S3, S4a, S4b of SURVEY.md 8(a)) for band
// limits whose working set fits shared memory.  Same mathematics as onsite_generic.cu:
//   Legendre synthesis (Eq.(36)) -> phi synthesis (Eq.(37) :327) -> pointwise product
//   (even channels, Eq.(38) :332) or surface-curl pairing (odd channels, Eq.(11) :107, theta-form) ->
//   inverse phi transform (Eq.(39) :339) -> Gauss-Legendre analysis (Eq.(40) :342),
// with the grid fields in registers only.  What differs is the mapping to the machine:
//   * lane = column: a CTA works on groups of 32 (atom, rank-channel) columns; every shared-memory array
//     has the column as its fastest index (or an odd row stride), so all accesses are conflict-free;
//   * packed FP32 FMAs (FFMA2, fma.rn.f32x2; 65 TFLOP/s measured against 57 for scalar FFMA): pairs are
//     (+m,-m) rows, (A,B) factors or (d_theta, d_phi) components.  Where the table value is common to both
//     halves it is a plain scalar: FFMA2 takes a 32-bit register broadcast to both lanes (SASS `R.F32`), so
//     one 128-bit broadcast load feeds four packed FMAs; only the odd stage A needs interleaved pairs;
//   * warps of a CTA split each stage by a static, host-computed schedule (longest-processing-time
//     assignment of the ragged per-m work), CTAs are persistent over column groups and prefetch the
//     next group's coefficients with TMA bulk copies while computing.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <mutex>

#include "onsite_core.cuh"

namespace cgtp {

struct CorePlan {
    int dev;  // CUDA device ordinal of `blob`
    int lmax, lmax_out;
    bool odd;
    bool wide;  // 8-warp CTAs where the on-site kernel wants them (band limit 8, odd channels)
    CoreTab tab;
    const void* blob;  // device
    std::vector<float> QF, QI;  // host copies of the azimuthal tables (kernel parameter CoreQParam)
};

// Host: packed tables + static schedules
// ------------------------------------------------------------------------------------------------
void lpt_assign(const std::vector<std::pair<int, int>>& items /* (cost, id) */, int NW,
                std::vector<std::vector<int>>& out, int* makespan)
{
    std::vector<std::pair<int, int>> it = items;
    std::stable_sort(it.begin(), it.end(), [](const std::pair<int, int>& a, const std::pair<int, int>& b) { return a.first > b.first; });
    std::vector<int> load(NW, 0);
    out.assign(NW, {});
    for (auto& x : it) {
        int w = 0;
        for (int k = 1; k < NW; ++k)
            if (load[k] < load[w]) w = k;
        load[w] += x.first;
        out[w].push_back(x.second);
    }
    *makespan = *std::max_element(load.begin(), load.end());
}

void stage_items(const Plan* p, bool odd, std::vector<std::pair<int, int>> (&items)[3])
{
    const int LB = p->LB;
    // stage A: cost ~ number of l terms (rows above lmax are zero-filled: cost 1).  even: one item per m <= LB
    // (both factors at once, they share the table loads); odd: one item per (m, factor), id = 2 m + factor
    for (int m = 0; m <= LB; ++m) {
        const int cost = m <= p->lmax ? 2 * (p->lmax - m + 1) + 1 : 1;
        if (!odd) {
            items[0].push_back({cost, m});
        } else {
            items[0].push_back({cost, 2 * m});
            items[0].push_back({cost, 2 * m + 1});
        }
    }
    // stage B: one item per grid row of a row block, equal cost (the kernel deals them round-robin)
    // (core_split: two half-rows per grid row)
    const int rows = (LB <= 8 ? p->U : 2 * core_ub(LB, odd)) * (core_split(LB, odd) ? 2 : 1);
    for (int u = 0; u < rows; ++u) items[1].push_back({4, u});
    // stage C: one item per m <= lmax_out
    for (int m = 0; m <= p->lmax_out; ++m) items[2].push_back({(p->lmax_out - m + 1) + 1, m});
}

static std::mutex g_core_mu;
static std::vector<CorePlan*> g_core_plans;

static size_t core_smem_bytes(const Plan* p, bool odd, const CoreTab& t, bool dbl)
{
    const int MR = 2 * p->LB + 1;
    const size_t gw = core_gw(p->LB, odd);
    const size_t hs = (size_t)2 * gw * onsite_fast_hstride(p) * 4;
    const size_t f = (size_t)(odd ? 4 : 2) * MR * (2 * core_ub(p->LB, odd)) * gw * 4;
    const size_t ts = gw * onsite_fast_tstride(p) * 4;
    return 64 + t.bytes + (dbl ? 2 : 1) * hs + f + ts;
}

void core_host_tables(const Plan* p, bool odd, CoreTab& t, std::vector<float>& TA, std::vector<float>& WP,
                      std::vector<float>& QF, std::vector<float>& QI)
{
    const int LB = p->LB, U = p->U, Uh = p->Uh, V = p->V;
    const int LL = LB + 1;
    const int MR = 2 * LB + 1;
    t.UP2 = round_up(core_uhmax(LB), 2);
    t.UP4 = round_up(core_uhmax(LB), 4);
    t.QFS = round_up(MR, 4);
    t.SOFF = round_up(LB + 1, 2);
    t.QIS = round_up(t.SOFF + LB, 4);
    const int ntri = (LB + 1) * (LB + 2) / 2;

    std::vector<double> x, w, P;
    gauss_legendre(U, x, w);
    legendre_values(U, LB, x, P);
    auto at = [&](int u, int l, int m) -> double { return P[((size_t)u * LL + l) * LL + m]; };

    TA.assign((size_t)ntri * (odd ? t.UP2 * 2 : t.UP4), 0.f);
    WP.assign((size_t)ntri * t.UP4, 0.f);
    for (int u = 0; u < Uh; ++u) {
        const double ct = x[u], st = std::sqrt(1.0 - ct * ct);
        const double wu = w[u] * ((U % 2 && u == Uh - 1) ? 0.5 : 1.0);
        for (int l = 0; l <= LB; ++l)
            for (int m = 0; m <= l; ++m) {
                const double pv = at(u, l, m);
                const double pm1 = (l - 1 >= m) ? at(u, l - 1, m) : 0.0;
                const double c = (l > 0) ? std::sqrt((2.0 * l + 1.0) * ((double)l * l - (double)m * m) / (2.0 * l - 1.0)) : 0.0;
                const double dth = (l * ct * pv - c * pm1) / st;
                if (!odd) {
                    TA[(size_t)tri_index(l, m) * t.UP4 + u] = (float)pv;
                } else {
                    const size_t k = ((size_t)tri_index(l, m) * t.UP2 + u) * 2;
                    TA[k] = (float)dth;
                    TA[k + 1] = (float)(m * pv / st);
                }
                WP[(size_t)tri_index(l, m) * t.UP4 + u] = (float)(wu * pv);
            }
    }
    // Azimuthal tables on the padded grid V4 = V rounded up to a multiple of 4 (exact as well, R8):
    // row vq = 0..V4/4 serves the four azimuths phi, -phi, pi - phi, pi + phi (quarter-wave folding); rows 0 and
    // V4/4 describe two distinct points each, visited twice -> half weight.
    const int V4 = round_up(V, 4), NQ = V4 / 4 + 1;
    QF.assign((size_t)NQ * t.QFS, 0.f);
    QI.assign((size_t)NQ * t.QIS, 0.f);
    for (int v = 0; v < NQ; ++v) {
        const double ph = 2.0 * M_PI * v / V4;
        const double wv = (2.0 * M_PI / V4) * ((v == 0 || v == NQ - 1) ? 0.5 : 1.0);
        for (int m = 0; m <= LB; ++m) {
            const double qc = (m == 0) ? 1.0 : std::sqrt(2.0) * std::cos(m * ph);
            const double qs = (m == 0) ? 0.0 : std::sqrt(2.0) * std::sin(m * ph);
            QF[(size_t)v * t.QFS + m] = (float)qc;
            QI[(size_t)v * t.QIS + m] = (float)(wv * qc);
            if (m > 0) {
                QF[(size_t)v * t.QFS + LB + m] = (float)qs;
                QI[(size_t)v * t.QIS + t.SOFF + m - 1] = (float)(wv * qs);
            }
        }
    }
    t.NQ = NQ;
}

// wide: the plan of launch_onsite_fast (see the warp count below); the two-field core and the single-kernel step keep the
// heuristic's CTA size (8 warps cost the pooled core of the two-field step 69.0 -> 76.7 ms on the configs[4] graph)
static const CorePlan* get_core_plan(const Plan* p, bool odd, bool wide = false)
{
    wide = wide && p->LB == 8 && odd;
    std::lock_guard<std::mutex> lk(g_core_mu);
    for (CorePlan* c : g_core_plans)
        if (c->dev == p->dev && c->lmax == p->lmax && c->lmax_out == p->lmax_out && c->odd == odd && c->wide == wide) return c;

    const int LB = p->LB;
    CoreTab t;
    std::memset(&t, 0, sizeof t);
    std::vector<float> TA, WP, QF, QI;
    core_host_tables(p, odd, t, TA, WP, QF, QI);

    // schedules: choose the warp count with the best work efficiency
    std::vector<std::pair<int, int>> items[3];
    stage_items(p, odd, items);
    int bestNW = 4;
    double best = -1.0;
    const int NH = 32 / core_gw(LB, odd);  // workers (schedule slots) per warp
    for (int NW = 4; NW <= kMaxWarps; ++NW) {
        double total = 0.0, span = 0.0;
        for (int s = 0; s < 3; ++s) {
            std::vector<std::vector<int>> asg;
            int mk;
            lpt_assign(items[s], NW * NH, asg, &mk);
            // stage B dominates the run time: weight it by its real share of the FMA work
            const double wgt = (s == 1) ? 6.0 : 1.0;
            int tot = 0;
            for (auto& x2 : items[s]) tot += x2.first;
            total += wgt * tot;
            span += wgt * mk * NW * NH;
        }
        const double eff = total / span;
        if (eff > best + 1e-9) { best = eff; bestNW = NW; }
    }
    t.NW = bestNW;
    // where one CTA per SM is all that fits (band limit 16 odd: row blocks of eight) every grid row of a block gets its own
    // half-warp: more resident warps count for more than the balance of the per-m lists
    if (LB >= 16 && core_ub(LB, odd) >= 8) t.NW = std::min(kMaxWarps, 2 * core_ub(LB, odd) / NH);
    // band limit 8, odd channels: 14 grid rows per group = 16 half-warp workers in one round of stage B; the heuristic keeps
    // 4 warps (two rounds, the same efficiency on paper), which leaves 8 warps per SM (two 93 KB CTAs) and 42 % of the issue
    // slots used.  Measured (configs[3] lmax 8, odd core): 4 / 6 / 8 warps 374 / 362 / 343 us; 8 warps lose at band limit 12
    // (row blocks of four: half the workers idle in stage B, 1.10 -> 1.61 ms) and for the even channels (193 -> 263 us)
    if (wide) t.NW = kMaxWarps;
    if (core_split(LB, odd)) t.NW = 2 * (2 * core_ub(LB, odd)) / NH;  // every (grid row, half of the azimuth rows) has its own half-warp: one pass
    std::vector<std::vector<int>> asg[3];
    int maxi = 1;
    for (int s = 0; s < 3; ++s) {
        int mk;
        lpt_assign(items[s], t.NW * NH, asg[s], &mk);
        for (auto& a : asg[s]) maxi = std::max(maxi, (int)a.size());
    }
    t.MAXI = maxi;
    std::vector<int> sched((size_t)3 * kMaxWorkers + (size_t)3 * kMaxWorkers * maxi, 0);
    for (int s = 0; s < 3; ++s)
        for (int wi = 0; wi < t.NW * NH; ++wi) {
            sched[s * kMaxWorkers + wi] = (int)asg[s][wi].size();
            for (size_t k = 0; k < asg[s][wi].size(); ++k)
                sched[3 * kMaxWorkers + ((size_t)s * kMaxWorkers + wi) * maxi + k] = asg[s][wi][k];
        }

    // pack
    std::vector<unsigned char> blob;
    auto append = [&](const void* src, size_t bytes) {
        size_t off = blob.size();
        blob.resize(off + round_up((int)bytes, 16));
        std::memcpy(blob.data() + off, src, bytes);
        return (int)off;
    };
    t.ta = append(TA.data(), TA.size() * 4);
    t.wp = append(WP.data(), WP.size() * 4);
    t.qf = append(QF.data(), QF.size() * 4);
    t.qi = append(QI.data(), QI.size() * 4);
    t.sched = append(sched.data(), sched.size() * 4);
    t.bytes = (int)blob.size();

    void* d = nullptr;
    if (cudaMalloc(&d, blob.size()) != cudaSuccess ||
        cudaMemcpy(d, blob.data(), blob.size(), cudaMemcpyHostToDevice) != cudaSuccess) {
        set_error("onsite core plan: device upload failed: %s", cudaGetErrorString(cudaGetLastError()));
        return nullptr;
    }
    CorePlan* c = new CorePlan;
    c->dev = p->dev;
    c->lmax = p->lmax;
    c->lmax_out = p->lmax_out;
    c->odd = odd;
    c->wide = wide;
    c->tab = t;
    c->blob = d;
    c->QF = QF;
    c->QI = QI;
    g_core_plans.push_back(c);
    return c;
}
struct CoreArgs {
    CoreTab tab;
    const void* blob;
    const float* Ha;
    const float* Hb;
    float* T;
    long long ngroups;
    int lmax, lmax_out, U, Uh, Vh;
    int L2s, Lo2s;
    int dbl;                         // 1: two H buffers (prefetch during the whole group), 0: one
    int off_blob, off_hs, off_f, off_ts;  // byte offsets in dynamic shared memory
    int hs_bytes;                    // bytes of one H buffer (both factors)
    // Two-field coupling (Eq.(28)): column = edge * cpar + channel and factor 2 of edge e is the block of
    // sender send[e] in Hb [senders][cpar][L2s]; cpar is a multiple of the group width, so a group never straddles two
    // edges.  send == nullptr: factor 2 is indexed like factor 1.  status != nullptr: leave when *status != 0 (M0 found
    // the edge list invalid, so send[] may not be dereferenced).
    const long long* send;
    int cpar;
    const int32_t* status;
};

template <int LB, bool ODD, int UB = core_ub(LB, ODD), bool SPLIT = core_split(LB, ODD)>
__global__ void __launch_bounds__(32 * kMaxWarps) onsite_fast_kernel(CoreArgs a, const __grid_constant__ CoreQParam<LB> qp)
{
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int MR = 2 * LB + 1;
    constexpr int RB = 2 * UB;
    constexpr int GW = core_gw(LB, ODD), NH = 32 / GW;  // columns per group; schedule slots (workers) per warp
    constexpr bool TWO_TERM = ODD && LB >= 20;     // four coefficient vectors of 2 LB + 1 pairs exceed the registers
    uint64_t* bar_tab = reinterpret_cast<uint64_t*>(smem);
    uint64_t* bar_h = reinterpret_cast<uint64_t*>(smem + 16);  // [2]
    const unsigned char* blob = smem + a.off_blob;
    const float* ta = reinterpret_cast<const float*>(blob + a.tab.ta);
    const float* wp = reinterpret_cast<const float*>(blob + a.tab.wp);
    const float* qf = reinterpret_cast<const float*>(blob + a.tab.qf);
    const float* qi = reinterpret_cast<const float*>(blob + a.tab.qi);
    const int* sched = reinterpret_cast<const int*>(blob + a.tab.sched);
    float* F = reinterpret_cast<float*>(smem + a.off_f);
    float* Ts = reinterpret_cast<float*>(smem + a.off_ts);
    constexpr int plane = MR * RB * GW;

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, NW = blockDim.x >> 5;
    const int col = lane & (GW - 1);                 // column of the group this lane works on
    const int worker = warp * NH + lane / GW, nworkers = NW * NH;
    const int hfl = GW * a.L2s;  // floats of one factor's H block
    const uint32_t hbytes = (uint32_t)hfl * 4;

    auto load_h = [&](long long g, int buf) {
        float* dst = reinterpret_cast<float*>(smem + a.off_hs + (size_t)buf * a.hs_bytes);
        mbar_arrive_expect_tx(&bar_h[buf], 2 * hbytes);
        tma_load_span(dst, a.Ha + g * hfl, hbytes, &bar_h[buf]);
        const float* hb = a.Hb + g * hfl;
        if (a.send) {
            const long long c0 = g * GW, e = c0 / a.cpar;
            hb = a.Hb + ((size_t)a.send[e] * a.cpar + (size_t)(c0 - e * a.cpar)) * a.L2s;
        }
        tma_load_span(dst + hfl, hb, hbytes, &bar_h[buf]);
    };
    pdl_launch_dependents();
    if (a.status) {  // written by an earlier kernel of the stream: nothing may be read before the predecessor is done
        pdl_wait();
        if (*a.status != 0) return;
    }

    if (threadIdx.x == 0) {
        mbar_init(bar_tab, 1);
        mbar_init(&bar_h[0], 1);
        mbar_init(&bar_h[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    long long g = blockIdx.x;
    if (threadIdx.x == 0) {
        mbar_arrive_expect_tx(bar_tab, (uint32_t)a.tab.bytes);
        tma_load_span(smem + a.off_blob, a.blob, (uint32_t)a.tab.bytes, bar_tab);  // the plan's tables: independent
        pdl_wait();  // H is the predecessor's output (this thread issues every load of it; T is written after H arrived)
        if (g < a.ngroups) load_h(g, 0);
    }
    mbar_wait(bar_tab, 0);

    const int MAXI = a.tab.MAXI;
    const int na = sched[0 * kMaxWorkers + worker], nc = sched[2 * kMaxWorkers + worker];
    const int* ia = sched + 3 * kMaxWorkers + (0 * kMaxWorkers + worker) * MAXI;
    const int* ic = sched + 3 * kMaxWorkers + (2 * kMaxWorkers + worker) * MAXI;
    const int nblk = (a.Uh + UB - 1) / UB;
    const int e_equator = (a.U & 1) ? a.Uh - 1 : -1;  // odd U: the last northern node is the equator, its own mirror image

    int buf = 0;
    uint32_t phases = 0u;  // bit b = parity to wait for on bar_h[b]
    for (; g < a.ngroups; g += gridDim.x) {
        const long long gn = g + gridDim.x;
        if (a.dbl && threadIdx.x == 0 && gn < a.ngroups) load_h(gn, buf ^ 1);
        mbar_wait(&bar_h[buf], (phases >> buf) & 1u);
        phases ^= 1u << buf;
        const float* hs = reinterpret_cast<const float*>(smem + a.off_hs + (size_t)buf * a.hs_bytes);
        const float* ha = hs + col * a.L2s;
        const float* hb = hs + hfl + col * a.L2s;

        for (int blk = 0; blk < nblk; ++blk) {
            const int e0 = blk * UB;
            const int ne = (a.Uh - e0 < UB) ? (a.Uh - e0) : UB;
            const int eq = (e_equator >= e0 && e_equator < e0 + UB) ? e_equator - e0 : -1;

            // ---- stage A: Legendre synthesis of the block's rows
            for (int k = 0; k < na; ++k) {
                if (!ODD) {
                    stage_a_even<LB, UB, GW>(ta, a.tab.UP4, ha, hb, F, F + plane, ia[k], a.lmax, e0, ne, col);
                } else {
                    const int m = ia[k] >> 1, f = ia[k] & 1;
                    stage_a_odd<LB, UB, GW>(ta, a.tab.UP2, f ? hb : ha, F + (2 * f) * plane, F + (2 * f + 1) * plane, m,
                                            a.lmax, e0, ne, col);
                }
            }
            __syncthreads();
            if (!a.dbl && blk == nblk - 1 && threadIdx.x == 0 && gn < a.ngroups) load_h(gn, 0);

            // ---- stage B: one local grid row per worker pass (north rows 0..ne-1, south rows UB..UB+ne-1; the
            // equator's southern copy is skipped)
            if constexpr (SPLIT) {
                // two warps per grid row, each with half of the azimuth rows; one pass (NW * NH == 2 RB)
                const int nwh = NW >> 1, vh = warp / nwh;
                const int lr = (warp - vh * nwh) * NH + lane / GW;
                const int e = (lr < UB) ? lr : lr - UB;
                const bool act = lr < RB && e < ne && !(lr >= UB && e == eq);
                const int vqm = (a.Vh + 1) >> 1;
                if constexpr (TWO_TERM)
                    stage_b_two_term<LB, RB, GW, true>(qf, qi, a.tab.QFS, a.tab.QIS, a.tab.SOFF, F, plane, lr,
                                                       vh ? a.Vh : vqm, col, act, vh ? vqm : 0, vh);
                else
                    stage_b<LB, ODD, RB, GW, true>(qf, qi, a.tab.QFS, a.tab.QIS, a.tab.SOFF, F, plane, lr,
                                                   vh ? a.Vh : vqm, col, act, vh ? vqm : 0, vh);
            } else
            for (int lr = worker; lr < RB; lr += nworkers) {
                const int e = (lr < UB) ? lr : lr - UB;
                if (e >= ne || (lr >= UB && e == eq)) continue;
                if constexpr (TWO_TERM)
                    stage_b_two_term<LB, RB, GW>(qf, qi, a.tab.QFS, a.tab.QIS, a.tab.SOFF, F, plane, lr, a.Vh, col);
                else if constexpr (LB <= 12)
                    stage_b_p<LB, ODD, RB, GW>(qp, F, plane, lr, a.Vh, col);  // tables as constant-bank operands
                else  // the fully unrolled form outgrows the instruction cache at band limits 16 and 20 (measured slower)
                    stage_b<LB, ODD, RB, GW>(qf, qi, a.tab.QFS, a.tab.QIS, a.tab.SOFF, F, plane, lr, a.Vh, col);
            }
            // the previous group's bulk store must have finished reading Ts before stage C rewrites it
            if (blk == 0 && threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
            __syncthreads();

            // ---- stage C: quadrature over the block's rows, accumulated over the blocks
            for (int k = 0; k < nc; ++k)
                stage_c<LB, UB, GW, SPLIT>(wp, a.tab.UP4, F, Ts + col * a.Lo2s, ic[k], a.lmax_out, e0, ne, eq, blk == 0, col,
                                           plane);
            if (blk == nblk - 1) fence_async_smem();
            __syncthreads();
        }
        if (threadIdx.x == 0) {
            tma_store_1d(a.T + g * GW * a.Lo2s, Ts, (uint32_t)(GW * a.Lo2s * 4));
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
        if (a.dbl) buf ^= 1;
    }
    if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// ------------------------------------------------------------------------------------------------
// Launch
// ------------------------------------------------------------------------------------------------

constexpr size_t kSmemPerSm = 227 * 1024;

// 0 if the fast kernel cannot run this plan; otherwise the dynamic shared memory per CTA, with *dbl set.
static size_t core_config(const Plan* p, bool odd, const CorePlan* c, bool* dbl)
{
    const size_t two = core_smem_bytes(p, odd, c->tab, true), one = core_smem_bytes(p, odd, c->tab, false);
    // prefer double-buffered H when it does not cost a resident CTA
    const size_t ctas_two = kSmemPerSm / (two + 1024), ctas_one = kSmemPerSm / (one + 1024);
    if (ctas_one == 0) return 0;
    *dbl = (ctas_two == ctas_one);
    return *dbl ? two : one;
}

bool onsite_fast_supported(const Plan* p, bool odd)
{
    const CorePlan* c = get_core_plan(p, odd);
    if (!c) return false;
    bool dbl;
    return core_config(p, odd, c, &dbl) != 0;
}

template <int LB, bool ODD, int UB = core_ub(LB, ODD), bool SPLIT = core_split(LB, ODD)>
static int launch_fast_t(const Plan* p, const CorePlan* c, const float* Ha, const float* Hb, float* T, int64_t ncols,
                         cudaStream_t st, const int64_t* send = nullptr, int cpar = 0, const int32_t* status = nullptr)
{
    bool dbl = false;
    const size_t smem = core_config(p, ODD, c, &dbl);
    if (!smem) { set_error("onsite fast core: plan does not fit shared memory"); return CGTP_ERR_UNSUPPORTED; }
    CoreArgs a;
    a.tab = c->tab;
    a.blob = c->blob;
    a.Ha = Ha;
    a.Hb = Hb;
    a.T = T;
    a.send = reinterpret_cast<const long long*>(send);
    a.cpar = cpar;
    a.status = status;
    constexpr int GW = core_gw(LB, ODD);
    a.ngroups = (ncols + GW - 1) / GW;  // the caller pads the column count to a multiple of 32
    a.lmax = p->lmax;
    a.lmax_out = p->lmax_out;
    a.U = p->U;
    a.Uh = p->Uh;
    a.Vh = c->tab.NQ;  // rows of the quarter-wave azimuthal tables
    a.L2s = onsite_fast_hstride(p);
    a.Lo2s = onsite_fast_tstride(p);
    a.dbl = dbl ? 1 : 0;
    a.hs_bytes = 2 * GW * a.L2s * 4;
    a.off_blob = 64;
    a.off_hs = a.off_blob + c->tab.bytes;
    a.off_f = a.off_hs + (dbl ? 2 : 1) * a.hs_bytes;
    a.off_ts = a.off_f + (ODD ? 4 : 2) * (2 * LB + 1) * (2 * UB) * GW * 4;
    auto kern = onsite_fast_kernel<LB, ODD, UB, SPLIT>;
    CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    // persistent CTAs: exactly as many as are resident at once (shared memory and registers both count)
    int ctas_per_sm = 0;
    CGTP_CUDA_CHECK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas_per_sm, kern, 32 * c->tab.NW, smem));
    if (ctas_per_sm < 1) ctas_per_sm = 1;
    int64_t grid = (int64_t)num_sms() * ctas_per_sm;
    if (grid > a.ngroups) grid = a.ngroups;
    CoreQParam<LB> qp;
    std::memset(&qp, 0, sizeof qp);
    std::memcpy(qp.qf, c->QF.data(), std::min(sizeof qp.qf, c->QF.size() * sizeof(float)));
    std::memcpy(qp.qi, c->QI.data(), std::min(sizeof qp.qi, c->QI.size() * sizeof(float)));
    LaunchScope scope(ODD ? K_ONSITE_ODD : K_ONSITE_EVEN, st);
    CGTP_CUDA_CHECK(launch_pdl(kern, (unsigned)grid, 32u * c->tab.NW, smem, st, a, qp));
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

int launch_onsite_fast(const Plan* p, bool odd, const float* Ha, const float* Hb, float* T, int64_t ncols,
                       cudaStream_t st)
{
    if (ncols <= 0) return CGTP_OK;
    if (onsite_reg_supported(p, odd) && !(kernel_path() & PATH_SMEM_CORE))
        return launch_onsite_reg(p, odd, Ha, Hb, T, ncols, st, nullptr, 0, nullptr);
    const CorePlan* c = get_core_plan(p, odd, true);
    if (!c) return CGTP_ERR_CUDA;
    switch (p->LB) {
#define CGTP_CASE(B)                                                              \
    case B:                                                                       \
        return odd ? launch_fast_t<B, true>(p, c, Ha, Hb, T, ncols, st)           \
                   : launch_fast_t<B, false>(p, c, Ha, Hb, T, ncols, st);
        CGTP_CASE(1) CGTP_CASE(2) CGTP_CASE(3) CGTP_CASE(4) CGTP_CASE(5) CGTP_CASE(6) CGTP_CASE(8) CGTP_CASE(10)
        CGTP_CASE(12) CGTP_CASE(16) CGTP_CASE(20)
#undef CGTP_CASE
    }
    set_error("onsite fast core: no kernel for band limit %d", p->LB);
    return CGTP_ERR_UNSUPPORTED;
}

// ------------------------------------------------------------------------------------------------
// Two-field coupling with the neighbour sum ON THE GRID (Eq.(52) PAPER.md:415 for Eq.(28) :236): one work item = (receiver,
// group of GW rank channels).  The CTA walks the receiver's in-edges inside the chunk [e0, e1): per edge stage A of both
// factors (the edge field's block of Ha, the sender's block of Hn through the edge list, TMA double-buffered) and the
// forward half of stage B, whose quarter-wave combinations are summed over the edges in registers; then ONE inverse
// transform and ONE Legendre analysis per receiver, added to Tn (a segment continued in the next chunk adds its part
// there: fixed order, no floating-point atomics).  Against one full core pass per edge plus a pooling kernel this drops the
// per-edge inverse transform, the per-edge analysis and the T round trip.
// ------------------------------------------------------------------------------------------------
struct PoolArgs {
    CoreTab tab;
    const void* blob;
    const float* Ha;            // [e1 - e0][cpar][L2s]: projected edge field of the chunk
    const float* Hn;            // [senders][cpar][L2s]
    const long long* send;      // senders of the whole edge list
    const long long* row_ptr;   // [nodes + 1]
    float* Tn;                  // [nodes][cpar][Lo2s]
    const int32_t* status;
    long long nodes, e0, e1;
    int cpar, lmax, lmax_out, U, Uh, NQ, L2s, Lo2s;
    int off_blob, off_hs, off_f, off_ts, hs_bytes;
};

template <int LB, bool ODD>
__global__ void __launch_bounds__(32 * kMaxWarps) field_pool_core_kernel(PoolArgs a, const __grid_constant__ CoreQParam<LB> qp)
{
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int MR = 2 * LB + 1;
    constexpr int UB = core_ub(LB, ODD), RB = 2 * UB;
    constexpr int GW = core_gw(LB, ODD), NH = 32 / GW;
    constexpr int MAXR = (GW == 32) ? 3 : 2;  // grid rows per worker (host-checked)
    constexpr int NQM = CoreQParam<LB>::NQMAX;
    uint64_t* bar_tab = reinterpret_cast<uint64_t*>(smem);
    uint64_t* bar_h = reinterpret_cast<uint64_t*>(smem + 16);  // [2]
    const unsigned char* blob = smem + a.off_blob;
    const float* ta = reinterpret_cast<const float*>(blob + a.tab.ta);
    const float* wp = reinterpret_cast<const float*>(blob + a.tab.wp);
    const int* sched = reinterpret_cast<const int*>(blob + a.tab.sched);
    float* F = reinterpret_cast<float*>(smem + a.off_f);
    float* Ts = reinterpret_cast<float*>(smem + a.off_ts);
    constexpr int plane = MR * RB * GW;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, NW = blockDim.x >> 5;
    const int col = lane & (GW - 1);
    const int worker = warp * NH + lane / GW, nworkers = NW * NH;
    const int hfl = GW * a.L2s;
    const uint32_t hbytes = (uint32_t)hfl * 4;
    const int ngrp = a.cpar / GW;
    if (*a.status != 0) return;  // M0 flagged the edge list: send[] may not be dereferenced (Tn stays zero)

    if (tid == 0) {
        mbar_init(bar_tab, 1);
        mbar_init(&bar_h[0], 1);
        mbar_init(&bar_h[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) {
        mbar_arrive_expect_tx(bar_tab, (uint32_t)a.tab.bytes);
        tma_load_span(smem + a.off_blob, a.blob, (uint32_t)a.tab.bytes, bar_tab);
    }
    auto load_h = [&](long long e, int g, int buf) {
        float* dst = reinterpret_cast<float*>(smem + a.off_hs + (size_t)buf * a.hs_bytes);
        mbar_arrive_expect_tx(&bar_h[buf], 2 * hbytes);
        tma_load_span(dst, a.Ha + ((size_t)(e - a.e0) * a.cpar + (size_t)g * GW) * a.L2s, hbytes, &bar_h[buf]);
        tma_load_span(dst + hfl, a.Hn + ((size_t)a.send[e] * a.cpar + (size_t)g * GW) * a.L2s, hbytes, &bar_h[buf]);
    };
    mbar_wait(bar_tab, 0);

    const int MAXI = a.tab.MAXI;
    const int na = sched[0 * kMaxWorkers + worker], nc = sched[2 * kMaxWorkers + worker];
    const int* ia = sched + 3 * kMaxWorkers + (0 * kMaxWorkers + worker) * MAXI;
    const int* ic = sched + 3 * kMaxWorkers + (2 * kMaxWorkers + worker) * MAXI;
    const int ne = a.Uh;
    const int eq = (a.U & 1) ? a.Uh - 1 : -1;

    int buf = 0;
    uint32_t phases = 0u;
    const long long nitems = a.nodes * ngrp;
    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        const long long i = item / ngrp;
        const int g = (int)(item - i * ngrp);
        const long long lo = a.row_ptr[i] > a.e0 ? a.row_ptr[i] : a.e0;
        const long long hi = a.row_ptr[i + 1] < a.e1 ? a.row_ptr[i + 1] : a.e1;
        if (lo >= hi) continue;
        float2 acc[MAXR][NQM][2];
#pragma unroll
        for (int r = 0; r < MAXR; ++r)
#pragma unroll
            for (int v = 0; v < NQM; ++v) acc[r][v][0] = acc[r][v][1] = make_float2(0.f, 0.f);
        if (tid == 0) load_h(lo, g, buf);
        for (long long e = lo; e < hi; ++e) {
            if (tid == 0 && e + 1 < hi) load_h(e + 1, g, buf ^ 1);
            mbar_wait(&bar_h[buf], (phases >> buf) & 1u);
            phases ^= 1u << buf;
            const float* hs = reinterpret_cast<const float*>(smem + a.off_hs + (size_t)buf * a.hs_bytes);
            const float* ha = hs + col * a.L2s;
            const float* hb = hs + hfl + col * a.L2s;
            for (int k = 0; k < na; ++k) {
                if (!ODD) {
                    stage_a_even<LB, UB, GW>(ta, a.tab.UP4, ha, hb, F, F + plane, ia[k], a.lmax, 0, ne, col);
                } else {
                    const int m = ia[k] >> 1, f = ia[k] & 1;
                    stage_a_odd<LB, UB, GW>(ta, a.tab.UP2, f ? hb : ha, F + (2 * f) * plane, F + (2 * f + 1) * plane, m, a.lmax,
                                            0, ne, col);
                }
            }
            __syncthreads();
#pragma unroll
            for (int r = 0; r < MAXR; ++r) {
                const int lr = worker + r * nworkers;
                if (lr < RB) {
                    const int e_ = (lr < UB) ? lr : lr - UB;
                    if (!(e_ >= ne || (lr >= UB && e_ == eq)))
                        stage_b_fwd_p<LB, ODD, RB, GW>(qp, F, plane, lr, a.NQ, col, acc[r]);
                }
            }
            __syncthreads();  // F and this H buffer are free again
            buf ^= 1;
        }
        // one inverse transform and one analysis for the pooled grid of the receiver
#pragma unroll
        for (int r = 0; r < MAXR; ++r) {
            const int lr = worker + r * nworkers;
            if (lr < RB) {
                const int e_ = (lr < UB) ? lr : lr - UB;
                if (!(e_ >= ne || (lr >= UB && e_ == eq))) stage_b_inv_p<LB, RB, GW>(qp, acc[r], F, lr, a.NQ, col);
            }
        }
        __syncthreads();
        for (int k = 0; k < nc; ++k) stage_c<LB, UB, GW>(wp, a.tab.UP4, F, Ts + col * a.Lo2s, ic[k], a.lmax_out, 0, ne, eq, true, col);
        __syncthreads();
        {
            float* dst = a.Tn + ((size_t)i * a.cpar + (size_t)g * GW) * a.Lo2s;
            const int n = GW * a.Lo2s;
            for (int idx = tid; idx < n; idx += blockDim.x) dst[idx] += Ts[idx];
        }
        __syncthreads();
    }
}

template <int LB, bool ODD>
static int launch_pool_t(const Plan* p, const CorePlan* c, const float* Ha, const float* Hn, const int64_t* send,
                         const int64_t* row_ptr, int cpar, const int32_t* status, float* Tn, int64_t nodes, int64_t e0,
                         int64_t e1, cudaStream_t st, bool* handled)
{
    constexpr int GW = core_gw(LB, ODD), NH = 32 / GW, RB = 2 * core_ub(LB, ODD);
    constexpr int MAXR = (GW == 32) ? 3 : 2;
    *handled = false;
    if (cpar % GW != 0) return CGTP_OK;
    if ((RB + c->tab.NW * NH - 1) / (c->tab.NW * NH) > MAXR) return CGTP_OK;
    const size_t smem = core_smem_bytes(p, ODD, c->tab, true);
    if (smem + 1024 > kSmemPerSm) return CGTP_OK;
    PoolArgs a;
    a.tab = c->tab;
    a.blob = c->blob;
    a.Ha = Ha;
    a.Hn = Hn;
    a.send = reinterpret_cast<const long long*>(send);
    a.row_ptr = reinterpret_cast<const long long*>(row_ptr);
    a.Tn = Tn;
    a.status = status;
    a.nodes = nodes;
    a.e0 = e0;
    a.e1 = e1;
    a.cpar = cpar;
    a.lmax = p->lmax;
    a.lmax_out = p->lmax_out;
    a.U = p->U;
    a.Uh = p->Uh;
    a.NQ = c->tab.NQ;
    a.L2s = onsite_fast_hstride(p);
    a.Lo2s = onsite_fast_tstride(p);
    a.hs_bytes = 2 * GW * a.L2s * 4;
    a.off_blob = 64;
    a.off_hs = a.off_blob + c->tab.bytes;
    a.off_f = a.off_hs + 2 * a.hs_bytes;
    a.off_ts = a.off_f + (ODD ? 4 : 2) * (2 * LB + 1) * RB * GW * 4;
    auto kern = field_pool_core_kernel<LB, ODD>;
    CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int ctas_per_sm = 0;
    CGTP_CUDA_CHECK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas_per_sm, kern, 32 * c->tab.NW, smem));
    if (ctas_per_sm < 1) ctas_per_sm = 1;
    const int64_t nitems = nodes * (cpar / GW);
    int64_t grid = (int64_t)num_sms() * ctas_per_sm;
    if (grid > nitems) grid = nitems;
    CoreQParam<LB> qp;
    std::memset(&qp, 0, sizeof qp);
    std::memcpy(qp.qf, c->QF.data(), std::min(sizeof qp.qf, c->QF.size() * sizeof(float)));
    std::memcpy(qp.qi, c->QI.data(), std::min(sizeof qp.qi, c->QI.size() * sizeof(float)));
    *handled = true;
    LaunchScope scope(ODD ? K_ONSITE_ODD : K_ONSITE_EVEN, st);
    kern<<<(unsigned)grid, 32 * c->tab.NW, smem, st>>>(a, qp);
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

// Ha: projected edge field of the edges [e0, e1) (columns (e - e0) * cpar + k), Hn: projected node field, send / row_ptr: the
// whole receiver-sorted edge list; Tn[i] += analysis of the pooled product grids of receiver i's in-edges inside the chunk.
// *handled = false when the shape is outside the kernel's limits (band limit > 8, cpar not a multiple of the group width):
// the caller then runs the per-edge core and the pooling kernel.
int launch_field_pool_core(const Plan* p, bool odd, const float* Ha, const float* Hn, const int64_t* send,
                           const int64_t* row_ptr, int cpar, const int32_t* status, float* Tn, int64_t nodes, int64_t e0,
                           int64_t e1, cudaStream_t st, bool* handled)
{
    *handled = false;
    if (cpar <= 0 || nodes <= 0 || e1 <= e0 || p->LB > 8) return CGTP_OK;
    const CorePlan* c = get_core_plan(p, odd);
    if (!c) return CGTP_ERR_CUDA;
    switch (p->LB) {
#define CGTP_CASE(B)                                                                                              \
    case B:                                                                                                       \
        return odd ? launch_pool_t<B, true>(p, c, Ha, Hn, send, row_ptr, cpar, status, Tn, nodes, e0, e1, st, handled)  \
                   : launch_pool_t<B, false>(p, c, Ha, Hn, send, row_ptr, cpar, status, Tn, nodes, e0, e1, st, handled);
        CGTP_CASE(1) CGTP_CASE(2) CGTP_CASE(3) CGTP_CASE(4) CGTP_CASE(5) CGTP_CASE(6) CGTP_CASE(8)
#undef CGTP_CASE
    }
    return CGTP_OK;
}

// Factor 2 gathered through the edge list (two-field coupling): column e * cpar + k pairs Ha's column with the block
// of sender send[e] in Hn.  *handled = false when the group width does not divide cpar (the caller gathers into a
// dense Hb and uses launch_onsite_fast).
int launch_onsite_fast_gather(const Plan* p, bool odd, const float* Ha, const float* Hn, const int64_t* send, int cpar,
                              const int32_t* status, float* T, int64_t ncols, cudaStream_t st, bool* handled)
{
    *handled = false;
    if (cpar <= 0 || cpar % core_gw(p->LB, odd) != 0) return CGTP_OK;
    *handled = true;
    if (ncols <= 0) return CGTP_OK;
    const CorePlan* c = get_core_plan(p, odd);
    if (!c) return CGTP_ERR_CUDA;
    switch (p->LB) {
#define CGTP_CASE(B)                                                                                   \
    case B:                                                                                            \
        return odd ? launch_fast_t<B, true>(p, c, Ha, Hn, T, ncols, st, send, cpar, status)            \
                   : launch_fast_t<B, false>(p, c, Ha, Hn, T, ncols, st, send, cpar, status);
        CGTP_CASE(1) CGTP_CASE(2) CGTP_CASE(3) CGTP_CASE(4) CGTP_CASE(5) CGTP_CASE(6) CGTP_CASE(8) CGTP_CASE(10)
        CGTP_CASE(12) CGTP_CASE(16) CGTP_CASE(20)
#undef CGTP_CASE
    }
    set_error("onsite fast core: no kernel for band limit %d", p->LB);
    return CGTP_ERR_UNSUPPORTED;
}

}  // namespace cgtp
