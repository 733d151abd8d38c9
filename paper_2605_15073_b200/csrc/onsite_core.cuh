// onsite_core.cuh -- stage functions and packed tables of the fused on-site core (rows S2a, S2b, S3, S4a, S4b of
// SURVEY.md 8(a)), shared by the core-only kernel (onsite_core.cu) and the whole-step kernel (onsite_fused.cu).
// See onsite_core.cu for the mapping (lane = column, packed FP32 FMAs, static warp schedules).
#pragma once

#include <utility>
#include <vector>

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


__host__ __device__ constexpr int core_uhmax(int LB) { return ((3 * LB + 2) / 2 + 1) / 2; }
// Columns per group: 32 (lane = column) at the small band limits; 16 from band limit 8 up (and for the odd channels at
// 6), where a warp works on two schedule items at once, one per half-warp: twice as many schedule slots balance the
// ragged per-m work and halve the shared memory per group.  Measured (configs[3], core even / odd, 32 -> 16 columns):
// lmax 8: 226 / 527 -> 205 / 402 us; 12: 1.25 / 1.80 -> 0.67 / 1.15 ms; 16: 3.16 / 4.77 -> 2.04 / 3.80 ms (odd with
// four-node row blocks); 20 odd (four-node row blocks): 11.2 -> 6.0 ms; configs[1] odd 106 -> 97 us, even 56 -> 63 us
// (kept at 32); lmax 2 and 4 are slower with 16.
__host__ __device__ constexpr int core_gw(int LB, bool odd) { return (LB >= 8 || (LB == 6 && odd)) ? 16 : 32; }
// Northern nodes per row block of the fast kernel: all of them (one block) for band limits <= 8; four for the larger
// ones, except eight for the odd channels at 16 and the even channels at 20; the odd channels at 20 give every grid row
// of stage B to two warps (core_split, see stage_b).  At 16 / 20 one group's H, T and F planes leave room for ONE CTA per
// SM, and with four-node blocks that CTA had 4 warps (ncu: one warp per scheduler, issue slots 23-30 % used); blocks of
// eight run with 8 warps (one half-warp per grid row of the block).  Measured on configs[3], core even / odd in ms --
// lmax 16: blocks of 4: 1.62 / 3.75 (even: 2 CTAs x 4 warps), split: 2.32 / 3.12, blocks of 8 on 8 warps: 1.99 / 2.15;
// lmax 20: blocks of 4: 4.67 / 6.18, split: 3.37 / 5.13, blocks of 8 on 8 warps: 2.26 / does not fit.
__host__ __device__ constexpr int core_ub(int LB, bool odd) { return LB <= 8 ? core_uhmax(LB) : ((LB == 16 && odd) || (LB == 20 && !odd)) ? 8 : 4; }
__host__ __device__ constexpr bool core_split(int LB, bool odd) { return LB >= 20 && odd; }


// Host (onsite_core.cu): longest-processing-time assignment of (cost, id) items to NW workers.
void lpt_assign(const std::vector<std::pair<int, int>>& items, int NW, std::vector<std::vector<int>>& out, int* makespan);
// Host: the packed FP32 tables of one (plan, parity) -- stage A table TA, analysis table WP, forward / inverse azimuthal
// tables QF / QI -- and their strides in `t` (offsets and schedule fields of `t` are left to the caller).
void core_host_tables(const Plan* p, bool odd, CoreTab& t, std::vector<float>& TA, std::vector<float>& WP,
                      std::vector<float>& QF, std::vector<float>& QI);
// Host: work items (cost, id) of the three stages for one column group.
void stage_items(const Plan* p, bool odd, std::vector<std::pair<int, int>> (&items)[3]);

// ------------------------------------------------------------------------------------------------
// Device
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float2 ffma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 fadd2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 fsub2(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }


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
// The azimuthal tables of stage B as a kernel parameter (constant bank): with the row loop fully unrolled every table
// index is a compile-time constant and the values are operands of the FMAs (uniform registers filled by LDCU), instead
// of 128-bit broadcast loads from shared memory, which cost two shared-memory wavefronts each -- the shared-memory pipe,
// not the FMA pipe, bound this stage (ncu: 75 % of the wavefront peak against 52 % FMA-pipe cycles).
template <int LB>
struct CoreQParam {
    static constexpr int QFS = round_up(2 * LB + 1, 4);
    static constexpr int SOFF = round_up(LB + 1, 2);
    static constexpr int QIS = round_up(SOFF + LB, 4);
    static constexpr int NQMAX = round_up(3 * LB + 1, 4) / 4 + 1;  // V4/4 + 1 at lmax = lmax_out = LB
    float qf[NQMAX * QFS], qi[NQMAX * QIS];
};

//
// SPLIT (band limits whose shared-memory footprint leaves room for one small CTA only): two warps share a grid row, each
// takes the azimuth rows [vq0, vq1) of the quarter-wave tables, and the two partial inverse transforms go to planes 0 and 1
// (stage C adds them).  Both planes are inputs of the partner warp, hence the CTA-wide barrier between the last load and
// the first store; `act` = this thread has a row (threads without one still take the barrier).
template <int LB, bool ODD, int RB, int GW, bool SPLIT = false>
__device__ __forceinline__ void stage_b(const float* __restrict__ qf, const float* __restrict__ qi, int QFS, int QIS,
                                        int SOFF, float* __restrict__ F, int plane_stride, int lr, int NQ, int lane,
                                        bool act = true, int vq0 = 0, int out_plane = 0)
{
    constexpr int MR = 2 * LB + 1;
    constexpr int NTC = (LB + 2) / 2;  // pairs of cos rows (m = 2k, 2k+1)
    constexpr int NTS = (LB + 1) / 2;  // pairs of sin rows (m = 2k+1, 2k+2)
    constexpr int NP = ODD ? 2 : 1;
    // f[k][r]: even: k = 0, pair (A, B); odd: k = 0 pair (A_theta, A_phi), k = 1 pair (B_theta, B_phi)
    float2 f[NP][MR];
    if (!SPLIT || act) {
#pragma unroll
        for (int r = 0; r < MR; ++r) {
            const int idx = (r * RB + lr) * GW + lane;
            f[0][r] = make_float2(F[idx], F[idx + plane_stride]);
            if (ODD) f[NP - 1][r] = make_float2(F[idx + 2 * plane_stride], F[idx + 3 * plane_stride]);
        }
    }
    float2 tc[NTC], ts[NTS > 0 ? NTS : 1];
#pragma unroll
    for (int k = 0; k < NTC; ++k) tc[k] = make_float2(0.f, 0.f);
#pragma unroll
    for (int k = 0; k < NTS; ++k) ts[k] = make_float2(0.f, 0.f);

#pragma unroll 2
    for (int vq = (SPLIT ? (act ? vq0 : NQ) : 0); vq < NQ; ++vq) {
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
    if (SPLIT) {
        __syncthreads();
        if (!act) return;
        F += (size_t)out_plane * plane_stride;
    }
#pragma unroll
    for (int m = 0; m <= LB; ++m) F[(m * RB + lr) * GW + lane] = (m & 1) ? tc[m / 2].y : tc[m / 2].x;
#pragma unroll
    for (int m = 1; m <= LB; ++m) F[((LB + m) * RB + lr) * GW + lane] = ((m - 1) & 1) ? ts[(m - 1) / 2].y : ts[(m - 1) / 2].x;
}

// Stage B of one (column, grid row) on registers.  f[k][r]: coefficient rows r = m (cosine, 0..LB), LB + m (sine); even
// channels: k = 0, pair (A, B); odd channels: PAIR_AB = false: f[0] = (A_theta, A_phi), f[1] = (B_theta, B_phi);
// PAIR_AB = true: f[0] = (A_theta, B_theta), f[1] = (A_phi, B_phi).  Result: tc[k] = cosine rows (m = 2k, 2k+1),
// ts[k] = sine rows (m = 2k+1, 2k+2), ADDED to the caller's values.  Fully unrolled over the largest table of the band
// limit: every table index is a compile-time constant, the values are constant-bank / uniform-register operands.
template <int LB, bool ODD, bool PAIR_AB = false>
__device__ __forceinline__ void stage_b_regs(const CoreQParam<LB>& qp, const float2 (&f)[ODD ? 2 : 1][2 * LB + 1], int NQ,
                                             float2 (&tc)[(LB + 2) / 2], float2 (&ts)[(LB + 1) / 2 > 0 ? (LB + 1) / 2 : 1])
{
    constexpr int MR = 2 * LB + 1;
    constexpr int NTC = (LB + 2) / 2;  // pairs of cos rows (m = 2k, 2k+1)
    constexpr int NTS = (LB + 1) / 2;  // pairs of sin rows (m = 2k+1, 2k+2)
    constexpr int NP = ODD ? 2 : 1;
    constexpr int QFS = CoreQParam<LB>::QFS, QIS = CoreQParam<LB>::QIS, SOFF = CoreQParam<LB>::SOFF;
#pragma unroll
    for (int vq = 0; vq < CoreQParam<LB>::NQMAX; ++vq) {
        if (vq >= NQ) break;
        float2 Ce[NP], Co[NP], Se[NP], So[NP];
#pragma unroll
        for (int k = 0; k < NP; ++k) Ce[k] = Co[k] = Se[k] = So[k] = make_float2(0.f, 0.f);
#pragma unroll
        for (int r = 0; r < MR; r += 4) {
            const float qv[4] = {qp.qf[vq * QFS + r], qp.qf[vq * QFS + r + 1], qp.qf[vq * QFS + r + 2], qp.qf[vq * QFS + r + 3]};
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
        } else if (!PAIR_AB) {
            // Eq.(11): {A,B} = A_theta B_phi - A_phi B_theta  (A factor 1, B factor 2)
            s1 = fmaf(g1[0].x, g1[NP - 1].y, -g1[0].y * g1[NP - 1].x);
            s2 = fmaf(g2[0].x, g2[NP - 1].y, -g2[0].y * g2[NP - 1].x);
            s3 = fmaf(g3[0].x, g3[NP - 1].y, -g3[0].y * g3[NP - 1].x);
            s4 = fmaf(g4[0].x, g4[NP - 1].y, -g4[0].y * g4[NP - 1].x);
        } else {
            s1 = fmaf(g1[0].x, g1[NP - 1].y, -g1[NP - 1].x * g1[0].y);
            s2 = fmaf(g2[0].x, g2[NP - 1].y, -g2[NP - 1].x * g2[0].y);
            s3 = fmaf(g3[0].x, g3[NP - 1].y, -g3[NP - 1].x * g3[0].y);
            s4 = fmaf(g4[0].x, g4[NP - 1].y, -g4[NP - 1].x * g4[0].y);
        }
        const float A = s1 + s2, B = s3 + s4, Cd = s1 - s2, D = s4 - s3;
        const float2 mc = make_float2(A + B, A - B);    // cosine rows: (even m, odd m)
        const float2 ms = make_float2(Cd - D, Cd + D);  // sine rows:   (odd m, even m)
#pragma unroll
        for (int k = 0; k < NTC; ++k)
            tc[k] = ffma2(make_float2(qp.qi[vq * QIS + 2 * k], qp.qi[vq * QIS + 2 * k + 1]), mc, tc[k]);
#pragma unroll
        for (int k = 0; k < NTS; ++k)
            ts[k] = ffma2(make_float2(qp.qi[vq * QIS + SOFF + 2 * k], qp.qi[vq * QIS + SOFF + 2 * k + 1]), ms, ts[k]);
    }
}

template <int LB, bool ODD, int RB, int GW>
__device__ __forceinline__ void stage_b_p(const CoreQParam<LB>& qp, float* __restrict__ F, int plane_stride, int lr, int NQ,
                                          int lane)
{
    constexpr int MR = 2 * LB + 1;
    constexpr int NTC = (LB + 2) / 2, NTS = (LB + 1) / 2;
    constexpr int NP = ODD ? 2 : 1;
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
    stage_b_regs<LB, ODD>(qp, f, NQ, tc, ts);
#pragma unroll
    for (int m = 0; m <= LB; ++m) F[(m * RB + lr) * GW + lane] = (m & 1) ? tc[m / 2].y : tc[m / 2].x;
#pragma unroll
    for (int m = 1; m <= LB; ++m) F[((LB + m) * RB + lr) * GW + lane] = ((m - 1) & 1) ? ts[(m - 1) / 2].y : ts[(m - 1) / 2].x;
}

// Stage B split in two for sums of products over several (factor 1, factor 2) pairs before ONE inverse transform (the
// neighbour sum on the grid of Eq.(52) PAPER.md:415 for the two-field coupling Eq.(28): the product grids of a receiver's
// in-edges are pooled before the analysis).  stage_b_fwd_p: forward transform and product of one grid row, the four
// quarter-wave combinations of every table row ADDED to acc[vq] = (mc, ms); stage_b_inv_p: inverse transform of the
// accumulated combinations into plane 0 of F.  Same arithmetic as stage_b_p, which is fwd + inv on a zero accumulator.
template <int LB, bool ODD, int RB, int GW>
__device__ __forceinline__ void stage_b_fwd_p(const CoreQParam<LB>& qp, const float* __restrict__ F, int plane_stride, int lr,
                                              int NQ, int lane, float2 (&acc)[CoreQParam<LB>::NQMAX][2])
{
    constexpr int MR = 2 * LB + 1;
    constexpr int NP = ODD ? 2 : 1;
    float2 f[NP][MR];
#pragma unroll
    for (int r = 0; r < MR; ++r) {
        const int idx = (r * RB + lr) * GW + lane;
        f[0][r] = make_float2(F[idx], F[idx + plane_stride]);
        if (ODD) f[NP - 1][r] = make_float2(F[idx + 2 * plane_stride], F[idx + 3 * plane_stride]);
    }
    constexpr int QFS = CoreQParam<LB>::QFS;
#pragma unroll
    for (int vq = 0; vq < CoreQParam<LB>::NQMAX; ++vq) {
        if (vq >= NQ) break;
        float2 Ce[NP], Co[NP], Se[NP], So[NP];
#pragma unroll
        for (int k = 0; k < NP; ++k) Ce[k] = Co[k] = Se[k] = So[k] = make_float2(0.f, 0.f);
#pragma unroll
        for (int rr = 0; rr < MR; ++rr) {
            const float qv = qp.qf[vq * QFS + rr];
            const float2 q2 = make_float2(qv, qv);
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
        float2 g1[NP], g2[NP], g3[NP], g4[NP];
#pragma unroll
        for (int k = 0; k < NP; ++k) {
            const float2 P = fadd2(Ce[k], Co[k]), Q = fsub2(Ce[k], Co[k]);
            const float2 R = fadd2(Se[k], So[k]), T = fsub2(Se[k], So[k]);
            g1[k] = fadd2(P, R);
            g2[k] = fsub2(P, R);
            g4[k] = fadd2(Q, T);
            g3[k] = fsub2(Q, T);
        }
        float s1, s2, s3, s4;
        if (!ODD) {
            s1 = g1[0].x * g1[0].y;
            s2 = g2[0].x * g2[0].y;
            s3 = g3[0].x * g3[0].y;
            s4 = g4[0].x * g4[0].y;
        } else {
            s1 = fmaf(g1[0].x, g1[NP - 1].y, -g1[0].y * g1[NP - 1].x);
            s2 = fmaf(g2[0].x, g2[NP - 1].y, -g2[0].y * g2[NP - 1].x);
            s3 = fmaf(g3[0].x, g3[NP - 1].y, -g3[0].y * g3[NP - 1].x);
            s4 = fmaf(g4[0].x, g4[NP - 1].y, -g4[0].y * g4[NP - 1].x);
        }
        const float A = s1 + s2, B = s3 + s4, Cd = s1 - s2, D = s4 - s3;
        acc[vq][0] = fadd2(acc[vq][0], make_float2(A + B, A - B));    // cosine rows: (even m, odd m)
        acc[vq][1] = fadd2(acc[vq][1], make_float2(Cd - D, Cd + D));  // sine rows:   (odd m, even m)
    }
}

template <int LB, int RB, int GW>
__device__ __forceinline__ void stage_b_inv_p(const CoreQParam<LB>& qp, const float2 (&acc)[CoreQParam<LB>::NQMAX][2],
                                              float* __restrict__ F, int lr, int NQ, int lane)
{
    constexpr int NTC = (LB + 2) / 2, NTS = (LB + 1) / 2;
    constexpr int QIS = CoreQParam<LB>::QIS, SOFF = CoreQParam<LB>::SOFF;
    float2 tc[NTC], ts[NTS > 0 ? NTS : 1];
#pragma unroll
    for (int k = 0; k < NTC; ++k) tc[k] = make_float2(0.f, 0.f);
#pragma unroll
    for (int k = 0; k < NTS; ++k) ts[k] = make_float2(0.f, 0.f);
#pragma unroll
    for (int vq = 0; vq < CoreQParam<LB>::NQMAX; ++vq) {
        if (vq >= NQ) break;
#pragma unroll
        for (int k = 0; k < NTC; ++k)
            tc[k] = ffma2(make_float2(qp.qi[vq * QIS + 2 * k], qp.qi[vq * QIS + 2 * k + 1]), acc[vq][0], tc[k]);
#pragma unroll
        for (int k = 0; k < NTS; ++k)
            ts[k] = ffma2(make_float2(qp.qi[vq * QIS + SOFF + 2 * k], qp.qi[vq * QIS + SOFF + 2 * k + 1]), acc[vq][1], ts[k]);
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
template <int LB, int RB, int GW, bool SPLIT = false>
__device__ __forceinline__ void stage_b_two_term(const float* __restrict__ qf, const float* __restrict__ qi, int QFS,
                                                 int QIS, int SOFF, float* __restrict__ F, int plane_stride, int lr,
                                                 int NQ, int lane, bool act = true, int vq0 = 0, int out_plane = 0)
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
        if (!SPLIT || act) {
#pragma unroll
            for (int r = 0; r < MR; ++r) {
                const int idx = (r * RB + lr) * GW + lane;
                f[r] = make_float2(F[idx + pa * plane_stride], F[idx + pb * plane_stride]);
            }
        }
#pragma unroll 2
        for (int vq = (SPLIT ? (act ? vq0 : NQ) : 0); vq < NQ; ++vq) {
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
    if (SPLIT) {
        __syncthreads();
        if (!act) return;
        F += (size_t)out_plane * plane_stride;
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
template <int LB, int UB, int GW, bool SPLIT = false>
__device__ __forceinline__ void stage_c(const float* __restrict__ wp, int UP4, const float* __restrict__ F,
                                        float* __restrict__ ts_col, int m, int lmax_out, int e0, int ne, int eq,
                                        bool first, int lane, int plane_stride = 0)
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
            if (SPLIT) {  // the two halves of the azimuth sum (stage_b, SPLIT)
                const float* F1 = F + plane_stride;
                n.x += F1[rn];
                s.x += F1[rs];
                if (m > 0) { n.y += F1[rn + off]; s.y += F1[rs + off]; }
            }
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

}  // namespace cgtp
