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

#include "sht.cuh"

namespace cgtp {

constexpr int kMaxWarps = 8;
constexpr int kMaxWorkers = 16;  // schedule slots: warps, or half-warps when a group has 16 columns

// Byte offsets (multiples of 16) into the packed table blob of one (plan, parity).
struct CoreTab {
    int ta;     // stage A: even [tri(l,m)][UP4] float P~; odd [tri(l,m)][UP2] float2 (d_theta P~, m P~/sin theta)
    int wp;     // stage C: [tri(l,m)][UP4] float w P~, equator row halved
    int qf;     // stage B forward: [NQ][QFS] float; entry r<=LB: cos row r, r>LB: sin row r-LB
    int qi;     // stage B inverse: [NQ][QIS] float, (2 pi/V4) q folded in; cos m at m, sin m at SOFF+m-1
    int sched;  // int: per stage s (A,B,C) and worker w: cnt[s][w] at s*kMaxWorkers+w, then items[s][w][MAXI]
    int bytes;
    int UP2, UP4, QFS, QIS, SOFF, MAXI;
    int NQ;     // rows of the azimuthal tables: V4/4 + 1, V4 = V rounded up to a multiple of 4
    int NW;
};

struct CorePlan {
    int dev;  // CUDA device ordinal of `blob`
    int lmax, lmax_out;
    bool odd;
    CoreTab tab;
    const void* blob;  // device
};

__host__ __device__ constexpr int core_uhmax(int LB) { return ((3 * LB + 2) / 2 + 1) / 2; }
// Columns per group: 32 (lane = column) at the small band limits; 16 from band limit 8 up (and for the odd channels at
// 6), where a warp works on two schedule items at once, one per half-warp: twice as many schedule slots balance the
// ragged per-m work and halve the shared memory per group.  Measured (configs[3], core even / odd, 32 -> 16 columns):
// lmax 8: 226 / 527 -> 205 / 402 us; 12: 1.25 / 1.80 -> 0.67 / 1.15 ms; 16: 3.16 / 4.77 -> 2.04 / 3.80 ms (odd with
// four-node row blocks); 20 odd (four-node row blocks): 11.2 -> 6.0 ms; configs[1] odd 106 -> 97 us, even 56 -> 63 us
// (kept at 32); lmax 2 and 4 are slower with 16.
__host__ __device__ constexpr int core_gw(int LB, bool odd) { return (LB >= 8 || (LB == 6 && odd)) ? 16 : 32; }
// Northern nodes per row block of the fast kernel: all of them (one block) for band limits <= 8; four for the
// larger ones.
__host__ __device__ constexpr int core_ub(int LB, bool odd) { return LB <= 8 ? core_uhmax(LB) : 4; }

// ------------------------------------------------------------------------------------------------
// Host: packed tables + static schedules
// ------------------------------------------------------------------------------------------------
static void lpt_assign(const std::vector<std::pair<int, int>>& items /* (cost, id) */, int NW,
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

static void stage_items(const Plan* p, bool odd, std::vector<std::pair<int, int>> (&items)[3])
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
    const int rows = LB <= 8 ? p->U : 2 * core_ub(LB, odd);
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

static const CorePlan* get_core_plan(const Plan* p, bool odd)
{
    std::lock_guard<std::mutex> lk(g_core_mu);
    for (CorePlan* c : g_core_plans)
        if (c->dev == p->dev && c->lmax == p->lmax && c->lmax_out == p->lmax_out && c->odd == odd) return c;

    const int LB = p->LB, U = p->U, Uh = p->Uh, V = p->V, Vh = p->Vh;
    const int LL = LB + 1;
    const int MR = 2 * LB + 1;
    CoreTab t;
    std::memset(&t, 0, sizeof t);
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

    std::vector<float> TA((size_t)ntri * (odd ? t.UP2 * 2 : t.UP4), 0.f), WP((size_t)ntri * t.UP4, 0.f);
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
    (void)Vh;
    std::vector<float> QF((size_t)NQ * t.QFS, 0.f), QI((size_t)NQ * t.QIS, 0.f);
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
    c->tab = t;
    c->blob = d;
    g_core_plans.push_back(c);
    return c;
}

// ------------------------------------------------------------------------------------------------
// Device
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float2 ffma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 fadd2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 fsub2(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }

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

// Grid rows are processed in blocks of UB northern nodes u' = e0 .. e0+UB-1 together with their mirror images
// U-1-u' (the pair shares one Legendre table row).  F holds one block: local row e (north) and UB+e (south),
// RB = 2 UB rows per coefficient row.  Band limits <= 8 use a single block (UB = all northern nodes); larger band
// limits use small blocks so that F fits shared memory, and stage C accumulates over the blocks.
//
// Stage A (row S2a), even channels.  Thread = (column, |m|): rows m (cos) and LB+m (sin) of both factors
// for the block's grid rows; pairs are (+m, -m), the table value is the broadcast scalar.
template <int LB, int UB, int GW>
__device__ __forceinline__ void stage_a_even(const float* __restrict__ ta, int UP4, const float* __restrict__ ha,
                                             const float* __restrict__ hb, float* __restrict__ Fa,
                                             float* __restrict__ Fb, int m, int lmax, int e0, int ne, int lane)
{
    constexpr int RB = 2 * UB;
    float2 acc[2][2][UB];
#pragma unroll
    for (int f = 0; f < 2; ++f)
#pragma unroll
        for (int par = 0; par < 2; ++par)
#pragma unroll
            for (int e = 0; e < UB; ++e) acc[f][par][e] = make_float2(0.f, 0.f);
    for (int l = m; l <= lmax; l += 2) {
#pragma unroll
        for (int par = 0; par < 2; ++par) {
            const int ll = l + par;
            if (ll > lmax) break;
            const float4* tab = reinterpret_cast<const float4*>(ta + (size_t)tri_index(ll, m) * UP4 + e0);
            const int ip = ll * ll + ll + m, im = ll * ll + ll - m;
            const float2 xa = make_float2(ha[ip], ha[im]);
            const float2 xb = make_float2(hb[ip], hb[im]);
#pragma unroll
            for (int e = 0; e < UB; e += 4) {
                const float4 t4 = tab[e / 4];
                const float tv[4] = {t4.x, t4.y, t4.z, t4.w};
#pragma unroll
                for (int h = 0; h < 4; ++h)
                    if (e + h < UB) {
                        acc[0][par][e + h] = ffma2(xa, make_float2(tv[h], tv[h]), acc[0][par][e + h]);
                        acc[1][par][e + h] = ffma2(xb, make_float2(tv[h], tv[h]), acc[1][par][e + h]);
                    }
            }
        }
    }
    // P~(-x) = (-1)^(l+m) P~(x): north = even + odd part, south = even - odd part
#pragma unroll
    for (int e = 0; e < UB; ++e) {
        if (e < ne) {
            const int rn = (m * RB + e) * GW + lane, rs = (m * RB + UB + e) * GW + lane;
            const int off = LB * RB * GW;
            const float2 na = fadd2(acc[0][0][e], acc[0][1][e]), sa = fsub2(acc[0][0][e], acc[0][1][e]);
            const float2 nb = fadd2(acc[1][0][e], acc[1][1][e]), sb = fsub2(acc[1][0][e], acc[1][1][e]);
            Fa[rn] = na.x; Fa[rs] = sa.x; Fb[rn] = nb.x; Fb[rs] = sb.x;
            if (m > 0) { Fa[rn + off] = na.y; Fa[rs + off] = sa.y; Fb[rn + off] = nb.y; Fb[rs + off] = sb.y; }
        }
    }
}

// Stage A, odd channels.  Table pairs are (d_theta P~, m P~/sin theta); accumulator pairs are the
// (theta, phi) components of the surface gradient.  The phi derivative swaps the cos and sin rows
// (PAPER.md:679): cos row m takes +m * (sine coefficient), sin row takes -m * (cosine coefficient).
// F planes: 2*f + 0 = d_theta, 2*f + 1 = (1/sin theta) d_phi of factor f.
template <int LB, int UB, int GW>
__device__ __forceinline__ void stage_a_odd(const float* __restrict__ ta, int UP2, const float* __restrict__ h,
                                            float* __restrict__ Fth, float* __restrict__ Fph, int m, int lmax, int e0,
                                            int ne, int lane)
{
    constexpr int RB = 2 * UB;
    float2 acc[2][2][UB];  // [row type: cos, sin][parity of l-m][u']
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
        for (int par = 0; par < 2; ++par)
#pragma unroll
            for (int e = 0; e < UB; ++e) acc[r][par][e] = make_float2(0.f, 0.f);
    for (int l = m; l <= lmax; l += 2) {
#pragma unroll
        for (int par = 0; par < 2; ++par) {
            const int ll = l + par;
            if (ll > lmax) break;
            const float4* tab = reinterpret_cast<const float4*>(ta + ((size_t)tri_index(ll, m) * UP2 + e0) * 2);
            const float hp = h[ll * ll + ll + m], hm = h[ll * ll + ll - m];
            const float2 xc = make_float2(hp, hm);   // cos row: d_theta from H[l,+m], d_phi from H[l,-m]
            const float2 xs = make_float2(hm, -hp);  // sin row: d_theta from H[l,-m], d_phi from -H[l,+m]
#pragma unroll
            for (int e = 0; e < UB; e += 2) {
                const float4 t4 = tab[e / 2];
                acc[0][par][e] = ffma2(make_float2(t4.x, t4.y), xc, acc[0][par][e]);
                acc[1][par][e] = ffma2(make_float2(t4.x, t4.y), xs, acc[1][par][e]);
                if (e + 1 < UB) {
                    acc[0][par][e + 1] = ffma2(make_float2(t4.z, t4.w), xc, acc[0][par][e + 1]);
                    acc[1][par][e + 1] = ffma2(make_float2(t4.z, t4.w), xs, acc[1][par][e + 1]);
                }
            }
        }
    }
    // d/dtheta flips the reflection parity; (1/sin) d_phi keeps it
#pragma unroll
    for (int e = 0; e < UB; ++e) {
        if (e < ne) {
            const int rn = (m * RB + e) * GW + lane, rs = (m * RB + UB + e) * GW + lane;
            const int off = LB * RB * GW;
            const float2 n0 = fadd2(acc[0][0][e], acc[0][1][e]), d0 = fsub2(acc[0][0][e], acc[0][1][e]);
            Fth[rn] = n0.x; Fth[rs] = -d0.x; Fph[rn] = n0.y; Fph[rs] = d0.y;
            if (m > 0) {
                const float2 n1 = fadd2(acc[1][0][e], acc[1][1][e]), d1 = fsub2(acc[1][0][e], acc[1][1][e]);
                Fth[rn + off] = n1.x; Fth[rs + off] = -d1.x; Fph[rn + off] = n1.y; Fph[rs + off] = d1.y;
            }
        }
    }
}

// Stage B (rows S2b + S3 + S4a) for one (column, grid row u): forward real DFT of the coefficient
// rows, product (even) or curl pairing (odd) at every azimuth, inverse real DFT -- all in registers.
// Quarter-wave folding: with Ce/Co the cosine sums over even/odd m and Se/So the sine sums, one table row
// gives the field at four azimuths,
//   f(phi) = Ce+Co+Se+So,  f(-phi) = Ce+Co-Se-So,  f(pi+phi) = Ce-Co+Se-So,  f(pi-phi) = Ce-Co-Se+So,
// and the inverse transform needs only  A+-B (cosine rows, even/odd m) and Cd+-D (sine rows) with
// A = s1+s2, B = s3+s4, Cd = s1-s2, D = s4-s3.  The result rows overwrite plane 0 in place.
template <int LB, bool ODD, int RB, int GW>
__device__ __forceinline__ void stage_b(const float* __restrict__ qf, const float* __restrict__ qi, int QFS, int QIS,
                                        int SOFF, float* __restrict__ F, int plane_stride, int lr, int NQ, int lane)
{
    constexpr int MR = 2 * LB + 1;
    constexpr int NTC = (LB + 2) / 2;  // pairs of cos rows (m = 2k, 2k+1)
    constexpr int NTS = (LB + 1) / 2;  // pairs of sin rows (m = 2k+1, 2k+2)
    constexpr int NP = ODD ? 2 : 1;
    // f[k][r]: even: k = 0, pair (A, B); odd: k = 0 pair (A_theta, A_phi), k = 1 pair (B_theta, B_phi)
    float2 f[NP][MR];
#pragma unroll
    for (int r = 0; r < MR; ++r) {
        const int idx = (r * RB + lr) * GW + lane;
        f[0][r] = make_float2(F[idx], F[idx + plane_stride]);
        if (ODD) f[NP - 1][r] = make_float2(F[idx + 2 * plane_stride], F[idx + 3 * plane_stride]);
    }
    float2 tc[NTC], ts[NTS > 0 ? NTS : 1];
#pragma unroll
    for (int k = 0; k < NTC; ++k) tc[k] = make_float2(0.f, 0.f);
#pragma unroll
    for (int k = 0; k < NTS; ++k) ts[k] = make_float2(0.f, 0.f);

#pragma unroll 2
    for (int vq = 0; vq < NQ; ++vq) {
        const float4* q4 = reinterpret_cast<const float4*>(qf + (size_t)vq * QFS);
        float2 Ce[NP], Co[NP], Se[NP], So[NP];
#pragma unroll
        for (int k = 0; k < NP; ++k) Ce[k] = Co[k] = Se[k] = So[k] = make_float2(0.f, 0.f);
#pragma unroll
        for (int r = 0; r < MR; r += 4) {
            const float4 t4 = q4[r / 4];
            const float qv[4] = {t4.x, t4.y, t4.z, t4.w};
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                const int rr = r + h;
                if (rr >= MR) break;
                const float2 q2 = make_float2(qv[h], qv[h]);
                const int m = (rr <= LB) ? rr : rr - LB;
#pragma unroll
                for (int k = 0; k < NP; ++k) {
                    if (rr <= LB) {
                        if (m & 1) Co[k] = ffma2(f[k][rr], q2, Co[k]);
                        else Ce[k] = ffma2(f[k][rr], q2, Ce[k]);
                    } else {
                        if (m & 1) So[k] = ffma2(f[k][rr], q2, So[k]);
                        else Se[k] = ffma2(f[k][rr], q2, Se[k]);
                    }
                }
            }
        }
        float2 g1[NP], g2[NP], g3[NP], g4[NP];
#pragma unroll
        for (int k = 0; k < NP; ++k) {
            const float2 P = fadd2(Ce[k], Co[k]), Q = fsub2(Ce[k], Co[k]);
            const float2 R = fadd2(Se[k], So[k]), T = fsub2(Se[k], So[k]);
            g1[k] = fadd2(P, R);  // phi
            g2[k] = fsub2(P, R);  // -phi
            g4[k] = fadd2(Q, T);  // pi + phi
            g3[k] = fsub2(Q, T);  // pi - phi
        }
        float s1, s2, s3, s4;
        if (!ODD) {
            // Eq.(38): A~ B~ at the four azimuths
            s1 = g1[0].x * g1[0].y;
            s2 = g2[0].x * g2[0].y;
            s3 = g3[0].x * g3[0].y;
            s4 = g4[0].x * g4[0].y;
        } else {
            // Eq.(11): {A,B} = A_theta B_phi - A_phi B_theta  (A factor 1, B factor 2)
            s1 = fmaf(g1[0].x, g1[NP - 1].y, -g1[0].y * g1[NP - 1].x);
            s2 = fmaf(g2[0].x, g2[NP - 1].y, -g2[0].y * g2[NP - 1].x);
            s3 = fmaf(g3[0].x, g3[NP - 1].y, -g3[0].y * g3[NP - 1].x);
            s4 = fmaf(g4[0].x, g4[NP - 1].y, -g4[0].y * g4[NP - 1].x);
        }
        const float A = s1 + s2, B = s3 + s4, Cd = s1 - s2, D = s4 - s3;
        const float2 mc = make_float2(A + B, A - B);    // cosine rows: (even m, odd m)
        const float2 ms = make_float2(Cd - D, Cd + D);  // sine rows:   (odd m, even m)
        const float2* qc2 = reinterpret_cast<const float2*>(qi + (size_t)vq * QIS);
        const float2* qs2 = reinterpret_cast<const float2*>(qi + (size_t)vq * QIS + SOFF);
#pragma unroll
        for (int k = 0; k < NTC; ++k) tc[k] = ffma2(qc2[k], mc, tc[k]);
#pragma unroll
        for (int k = 0; k < NTS; ++k) ts[k] = ffma2(qs2[k], ms, ts[k]);
    }
#pragma unroll
    for (int m = 0; m <= LB; ++m) F[(m * RB + lr) * GW + lane] = (m & 1) ? tc[m / 2].y : tc[m / 2].x;
#pragma unroll
    for (int m = 1; m <= LB; ++m) F[((LB + m) * RB + lr) * GW + lane] = ((m - 1) & 1) ? ts[(m - 1) / 2].y : ts[(m - 1) / 2].x;
}

// Stage B for odd channels at band limits whose four coefficient vectors do not fit the register file: the curl
// pairing {A,B} = A_theta B_phi - A_phi B_theta is evaluated as two product terms, each with its own forward
// transform of one (factor-1 field, factor-2 field) pair, sharing the inverse-transform accumulators by linearity.
// F planes: 0 = A_theta, 1 = A_phi, 2 = B_theta, 3 = B_phi.
template <int LB, int RB, int GW>
__device__ __forceinline__ void stage_b_two_term(const float* __restrict__ qf, const float* __restrict__ qi, int QFS,
                                                 int QIS, int SOFF, float* __restrict__ F, int plane_stride, int lr,
                                                 int NQ, int lane)
{
    constexpr int MR = 2 * LB + 1;
    constexpr int NTC = (LB + 2) / 2, NTS = (LB + 1) / 2;
    float2 tc[NTC], ts[NTS];
#pragma unroll
    for (int k = 0; k < NTC; ++k) tc[k] = make_float2(0.f, 0.f);
#pragma unroll
    for (int k = 0; k < NTS; ++k) ts[k] = make_float2(0.f, 0.f);
#pragma unroll 1
    for (int term = 0; term < 2; ++term) {
        const int pa = term ? 1 : 0, pb = term ? 2 : 3;
        const float sgn = term ? -1.f : 1.f;
        float2 f[MR];
#pragma unroll
        for (int r = 0; r < MR; ++r) {
            const int idx = (r * RB + lr) * GW + lane;
            f[r] = make_float2(F[idx + pa * plane_stride], F[idx + pb * plane_stride]);
        }
#pragma unroll 2
        for (int vq = 0; vq < NQ; ++vq) {
            const float4* q4 = reinterpret_cast<const float4*>(qf + (size_t)vq * QFS);
            float2 Ce = make_float2(0.f, 0.f), Co = Ce, Se = Ce, So = Ce;
#pragma unroll
            for (int r = 0; r < MR; r += 4) {
                const float4 t4 = q4[r / 4];
                const float qv[4] = {t4.x, t4.y, t4.z, t4.w};
#pragma unroll
                for (int h = 0; h < 4; ++h) {
                    const int rr = r + h;
                    if (rr >= MR) break;
                    const float2 q2 = make_float2(qv[h], qv[h]);
                    const int m = (rr <= LB) ? rr : rr - LB;
                    if (rr <= LB) {
                        if (m & 1) Co = ffma2(f[rr], q2, Co);
                        else Ce = ffma2(f[rr], q2, Ce);
                    } else {
                        if (m & 1) So = ffma2(f[rr], q2, So);
                        else Se = ffma2(f[rr], q2, Se);
                    }
                }
            }
            const float2 P = fadd2(Ce, Co), Q = fsub2(Ce, Co), R = fadd2(Se, So), T = fsub2(Se, So);
            const float2 g1 = fadd2(P, R), g2 = fsub2(P, R), g4 = fadd2(Q, T), g3 = fsub2(Q, T);
            const float s1 = sgn * (g1.x * g1.y), s2 = sgn * (g2.x * g2.y), s3 = sgn * (g3.x * g3.y),
                        s4 = sgn * (g4.x * g4.y);
            const float A = s1 + s2, B = s3 + s4, Cd = s1 - s2, D = s4 - s3;
            const float2 mc = make_float2(A + B, A - B), ms = make_float2(Cd - D, Cd + D);
            const float2* qc2 = reinterpret_cast<const float2*>(qi + (size_t)vq * QIS);
            const float2* qs2 = reinterpret_cast<const float2*>(qi + (size_t)vq * QIS + SOFF);
#pragma unroll
            for (int k = 0; k < NTC; ++k) tc[k] = ffma2(qc2[k], mc, tc[k]);
#pragma unroll
            for (int k = 0; k < NTS; ++k) ts[k] = ffma2(qs2[k], ms, ts[k]);
        }
    }
#pragma unroll
    for (int m = 0; m <= LB; ++m) F[(m * RB + lr) * GW + lane] = (m & 1) ? tc[m / 2].y : tc[m / 2].x;
#pragma unroll
    for (int m = 1; m <= LB; ++m) F[((LB + m) * RB + lr) * GW + lane] = ((m - 1) & 1) ? ts[(m - 1) / 2].y : ts[(m - 1) / 2].x;
}

// Stage C (row S4b, Eq.(40)): Gauss-Legendre quadrature over the block's grid rows for one
// (column, |m|); pairs are (+m, -m).  Ts: [32][Lo2s] staging for the bulk store; `first` = first block of the
// group (store), later blocks accumulate.  eq = index e of the equator row in this block (its mirror image is the
// row itself and stage B ran on the northern copy only), or -1.
template <int LB, int UB, int GW>
__device__ __forceinline__ void stage_c(const float* __restrict__ wp, int UP4, const float* __restrict__ F,
                                        float* __restrict__ ts_col, int m, int lmax_out, int e0, int ne, int eq,
                                        bool first, int lane)
{
    constexpr int RB = 2 * UB;
    float2 tp[UB], tm[UB];
#pragma unroll
    for (int e = 0; e < UB; ++e) {
        float2 n = make_float2(0.f, 0.f), s = make_float2(0.f, 0.f);
        if (e < ne) {
            const int rn = (m * RB + e) * GW + lane;
            const int rs = (e == eq) ? rn : (m * RB + UB + e) * GW + lane;
            const int off = LB * RB * GW;
            n.x = F[rn];
            s.x = F[rs];
            if (m > 0) { n.y = F[rn + off]; s.y = F[rs + off]; }
        }
        tp[e] = fadd2(n, s);
        tm[e] = fsub2(n, s);
    }
    for (int l = m; l <= lmax_out; l += 2) {
#pragma unroll
        for (int par = 0; par < 2; ++par) {
            const int ll = l + par;
            if (ll > lmax_out) break;
            const float4* tab = reinterpret_cast<const float4*>(wp + (size_t)tri_index(ll, m) * UP4 + e0);
            float2 a0 = make_float2(0.f, 0.f), a1 = make_float2(0.f, 0.f);
            if constexpr (UB == 2) {  // blocks of two rows start at even e0: 64-bit table loads
                const float2 t2 = *reinterpret_cast<const float2*>(tab);
                a0 = ffma2(par ? tm[0] : tp[0], make_float2(t2.x, t2.x), a0);
                a1 = ffma2(par ? tm[1] : tp[1], make_float2(t2.y, t2.y), a1);
            } else {
#pragma unroll
                for (int e = 0; e < UB; e += 4) {
                    const float4 t4 = tab[e / 4];
                    const float tv[4] = {t4.x, t4.y, t4.z, t4.w};
#pragma unroll
                    for (int h = 0; h < 4; ++h)
                        if (e + h < UB) {
                            const float2 x = par ? tm[e + h] : tp[e + h];
                            if (h & 1) a1 = ffma2(x, make_float2(tv[h], tv[h]), a1);
                            else a0 = ffma2(x, make_float2(tv[h], tv[h]), a0);
                        }
                }
            }
            const float2 r = fadd2(a0, a1);
            const int ip = ll * ll + ll + m, im = ll * ll + ll - m;
            ts_col[ip] = first ? r.x : ts_col[ip] + r.x;
            if (m > 0) ts_col[im] = first ? r.y : ts_col[im] + r.y;
        }
    }
}

template <int LB, bool ODD>
__global__ void __launch_bounds__(32 * kMaxWarps) onsite_fast_kernel(CoreArgs a)
{
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int MR = 2 * LB + 1;
    constexpr int UB = core_ub(LB, ODD), RB = 2 * UB;
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
    if (a.status && *a.status != 0) return;

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
        tma_load_span(smem + a.off_blob, a.blob, (uint32_t)a.tab.bytes, bar_tab);
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
            for (int lr = worker; lr < RB; lr += nworkers) {
                const int e = (lr < UB) ? lr : lr - UB;
                if (e >= ne || (lr >= UB && e == eq)) continue;
                if constexpr (TWO_TERM)
                    stage_b_two_term<LB, RB, GW>(qf, qi, a.tab.QFS, a.tab.QIS, a.tab.SOFF, F, plane, lr, a.Vh, col);
                else
                    stage_b<LB, ODD, RB, GW>(qf, qi, a.tab.QFS, a.tab.QIS, a.tab.SOFF, F, plane, lr, a.Vh, col);
            }
            // the previous group's bulk store must have finished reading Ts before stage C rewrites it
            if (blk == 0 && threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
            __syncthreads();

            // ---- stage C: quadrature over the block's rows, accumulated over the blocks
            for (int k = 0; k < nc; ++k)
                stage_c<LB, UB, GW>(wp, a.tab.UP4, F, Ts + col * a.Lo2s, ic[k], a.lmax_out, e0, ne, eq, blk == 0, col);
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

template <int LB, bool ODD>
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
    a.off_ts = a.off_f + (ODD ? 4 : 2) * (2 * LB + 1) * (2 * core_ub(LB, ODD)) * GW * 4;
    auto kern = onsite_fast_kernel<LB, ODD>;
    CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    // persistent CTAs: exactly as many as are resident at once (shared memory and registers both count)
    int ctas_per_sm = 0;
    CGTP_CUDA_CHECK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas_per_sm, kern, 32 * c->tab.NW, smem));
    if (ctas_per_sm < 1) ctas_per_sm = 1;
    int64_t grid = (int64_t)num_sms() * ctas_per_sm;
    if (grid > a.ngroups) grid = a.ngroups;
    LaunchScope scope(ODD ? K_ONSITE_ODD : K_ONSITE_EVEN, st);
    kern<<<(unsigned)grid, 32 * c->tab.NW, smem, st>>>(a);
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

int launch_onsite_fast(const Plan* p, bool odd, const float* Ha, const float* Hb, float* T, int64_t ncols,
                       cudaStream_t st)
{
    if (ncols <= 0) return CGTP_OK;
    const CorePlan* c = get_core_plan(p, odd);
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
