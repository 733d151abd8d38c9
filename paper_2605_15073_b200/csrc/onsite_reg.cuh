// onsite_reg.cuh -- the transform chain of ONE (atom, rank-channel) column on registers (rows S2a-S4b of SURVEY.md 8(a)),
// used by the register core (onsite_reg.cu; see there for the design).
#pragma once
#include "onsite_core.cuh"

namespace cgtp {

// entry t of the (l, m) triangle, t = l (l + 1) / 2 + m
__host__ __device__ constexpr int tri_l(int t) { int l = 0; while ((l + 1) * (l + 2) / 2 <= t) ++l; return l; }
__host__ __device__ constexpr int tri_m(int t) { return t - tri_l(t) * (tri_l(t) + 1) / 2; }

// Host: the Legendre row tables of one parity, [ntab][U][NT4] with NT4 = (LB+1)(LB+2)/2 rounded up to 4 and entry
// tri_index(l, m): even: P~_lm(x_u), w_u P~_lm(x_u); odd: d/dtheta P~_lm, m P~_lm / sin(theta), w_u P~_lm.  Rows above lmax
// (synthesis) / lmax_out (analysis) are zero.  Returns NT4.
int reg_host_tables(const Plan* p, bool odd, std::vector<float>& tab);

// All grid rows of one column.  tab0 / tab1 / tabw: the row tables in shared memory (warp-uniform broadcast loads);
// hh: the column's coefficients as (factor 1, factor 2) pairs when HREG, else they are re-read from ha / hb (shared memory,
// odd row stride) for every grid row; T: the column's output coefficients, accumulated over the rows (caller zeroes).
template <int LB, bool ODD, bool HREG>
__device__ __forceinline__ void reg_column_rows(const CoreQParam<LB>& qp, const float* __restrict__ tab0,
                                                const float* __restrict__ tab1, const float* __restrict__ tabw, int U, int NQ,
                                                int L2, const float* __restrict__ ha, const float* __restrict__ hb,
                                                const float2 (&hh)[HREG ? (LB + 1) * (LB + 1) : 1],
                                                float (&T)[(LB + 1) * (LB + 1)])
{
    constexpr int NT = (LB + 1) * (LB + 2) / 2, NT4 = round_up(NT, 4);
    constexpr int MR = 2 * LB + 1, NP = ODD ? 2 : 1;
    constexpr int NTC = (LB + 2) / 2, NTS = (LB + 1) / 2;
#pragma unroll 1
    for (int u = 0; u < U; ++u) {
        // ---- stage A: coefficient rows of grid row u.  Pairs are the two factors (A, B); table values are scalars.
        float2 f[NP][MR];
#pragma unroll
        for (int k = 0; k < NP; ++k)
#pragma unroll
            for (int r = 0; r < MR; ++r) f[k][r] = make_float2(0.f, 0.f);
#pragma unroll
        for (int j = 0; j < NT4; j += 4) {
            const float4 v0 = *reinterpret_cast<const float4*>(tab0 + u * NT4 + j);
            const float t0[4] = {v0.x, v0.y, v0.z, v0.w};
            float t1[4] = {0.f, 0.f, 0.f, 0.f};
            if (ODD) {
                const float4 v1 = *reinterpret_cast<const float4*>(tab1 + u * NT4 + j);
                t1[0] = v1.x; t1[1] = v1.y; t1[2] = v1.z; t1[3] = v1.w;
            }
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                if (j + h >= NT) break;
                const int l = tri_l(j + h), m = tri_m(j + h);
                const int ip = l * l + l + m, im = l * l + l - m;
                float2 xp, xm;
                if (HREG) {
                    xp = hh[ip];
                    xm = hh[im];
                } else {
                    const bool in = ip < L2;  // l <= lmax
                    xp = in ? make_float2(ha[ip], hb[ip]) : make_float2(0.f, 0.f);
                    xm = (in && m > 0) ? make_float2(ha[im], hb[im]) : xp;
                }
                const float2 p2 = make_float2(t0[h], t0[h]);
                f[0][m] = ffma2(xp, p2, f[0][m]);
                if (m > 0) f[0][LB + m] = ffma2(xm, p2, f[0][LB + m]);
                if (ODD && m > 0) {
                    // the phi derivative swaps the cosine and sine rows: cos row m takes
                    // +m (sine coefficient), sin row m takes -m (cosine coefficient)
                    f[NP - 1][m] = ffma2(xm, make_float2(t1[h], t1[h]), f[NP - 1][m]);
                    f[NP - 1][LB + m] = ffma2(xp, make_float2(-t1[h], -t1[h]), f[NP - 1][LB + m]);
                }
            }
        }
        // ---- stage B
        float2 tc[NTC], ts[NTS > 0 ? NTS : 1];
#pragma unroll
        for (int k = 0; k < NTC; ++k) tc[k] = make_float2(0.f, 0.f);
#pragma unroll
        for (int k = 0; k < NTS; ++k) ts[k] = make_float2(0.f, 0.f);
        stage_b_regs<LB, ODD, true>(qp, f, NQ, tc, ts);
        // ---- stage C: this row's term of the quadrature
#pragma unroll
        for (int j = 0; j < NT4; j += 4) {
            const float4 v = *reinterpret_cast<const float4*>(tabw + u * NT4 + j);
            const float wv[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                if (j + h >= NT) break;
                const int l = tri_l(j + h), m = tri_m(j + h);
                const float gc = (m & 1) ? tc[m / 2].y : tc[m / 2].x;
                T[l * l + l + m] = fmaf(wv[h], gc, T[l * l + l + m]);
                if (m > 0) {
                    const float gs = ((m - 1) & 1) ? ts[(m - 1) / 2].y : ts[(m - 1) / 2].x;
                    T[l * l + l - m] = fmaf(wv[h], gs, T[l * l + l - m]);
                }
            }
        }
    }
}

}  // namespace cgtp
