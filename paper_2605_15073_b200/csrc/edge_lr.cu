// edge_lr.cu -- rows M3 + M4 of SURVEY.md 8(a) with the paper's l1-DEPENDENT radial factor R~_{jicl1} (Eq.(46)
// PAPER.md:396): the edge field of channel c is  E_{e,c}(Omega) = sum_{l1} R~[e,c,l1] (2 l1+1)/(4 pi) P_{l1}(r_e . Omega)
// (Eq.(48), (50) :402-:408 through the addition theorem, R12 / 5.8), no longer a channel-independent field
// times a scalar.  The paper evaluates it as a per-(bond, channel) Legendre + Fourier transform -- the stage it measured
// as its heaviest (:687); here the zonal sum is evaluated directly at the grid points a thread owns:
//   * thread = (channel group, grid quad); the Legendre recurrence in t = r_e . Omega runs once per (edge, quad) in
//     registers and every degree's term is folded into the NA channels of the thread with their own R~[e,c,l1]
//     (staged per chunk of edges in shared memory), so no per-degree field is ever stored;
//   * the sender's VALUE grid is gathered for both parities; the odd channels pair it with (d_theta E, -(1/sin) d_phi E)
//     = (sum_l R~ c_l P'_l) (r_e . theta_hat, -r_e . phi_hat) into two pooled grids (by-parts form);
//   * neighbour sum in registers in input edge order: deterministic, no floating-point atomics.
// G: [n_send][Cpar][UVp]; S: even [nodes][Cpar][UVp], odd [nodes][Cpar][2][UVp]; edge_radial: [E][C][lmax+1].
#include <algorithm>

#include "sht.cuh"

namespace cgtp {

constexpr int LR_NT = 512;
constexpr int LR_EC = 32;    // edges per chunk (upper bound; the launcher picks EC <= LR_EC that fits shared memory)
constexpr int LR_LMAX = 24;  // recurrence coefficient table length

__device__ __forceinline__ float4 lr_ldg_stream(const float4* p)
{
    float4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w)
                 : "l"(p));
    return r;
}
__device__ __forceinline__ float4 lr_dot3(float ex, float ey, float ez, const float4& x, const float4& y, const float4& z)
{
    return make_float4(fmaf(ex, x.x, fmaf(ey, y.x, ez * z.x)), fmaf(ex, x.y, fmaf(ey, y.y, ez * z.y)),
                       fmaf(ex, x.z, fmaf(ey, y.z, ez * z.z)), fmaf(ex, x.w, fmaf(ey, y.w, ez * z.w)));
}
__device__ __forceinline__ void lr_axpy(float4& a, float s, const float4& v)
{
    a.x = fmaf(s, v.x, a.x); a.y = fmaf(s, v.y, a.y); a.z = fmaf(s, v.z, a.z); a.w = fmaf(s, v.w, a.w);
}
__device__ __forceinline__ void lr_fma4(float4& a, const float4& u, const float4& v)
{
    a.x = fmaf(u.x, v.x, a.x); a.y = fmaf(u.y, v.y, a.y); a.z = fmaf(u.z, v.z, a.z); a.w = fmaf(u.w, v.w, a.w);
}

template <bool ODD, int NA, int LB>
__global__ void __launch_bounds__(LR_NT, 1) edge_lr_kernel(Plan p, const float* __restrict__ G,
                                                          const int64_t* __restrict__ row_ptr,
                                                          const int64_t* __restrict__ snd,
                                                          const float* __restrict__ edge_vec,
                                                          const float* __restrict__ radial,
                                                          const int* __restrict__ perm_par, int Cpar, int C, int cb,
                                                          int nblk, int G_, int EC, float* __restrict__ S,
                                                          const int32_t* __restrict__ status)
{
    constexpr int NF = ODD ? 2 : 1;
    constexpr int NG = ODD ? 8 : 3;  // geometry fields: Omega_xyz (+ theta_hat_xyz, phi_hat_xy)
    extern __shared__ __align__(16) unsigned char smem_lr[];
    float4* Es = reinterpret_cast<float4*>(smem_lr);               // [LR_EC] unit vectors
    long long* Ss = reinterpret_cast<long long*>(Es + LR_EC);      // [EC] senders
    // the degree loop is unrolled to the kernel band limit LB >= lmax: recurrence coefficients are immediates and the
    // R~ rows are zero beyond lmax
    const int UVp = p.UVp, QP = UVp / 4, lmax = p.lmax, L1 = lmax + 1;
    constexpr int L1p = round_up(LB + 1, 4);
    float4* geo_s = reinterpret_cast<float4*>(Ss + LR_EC);         // [NG][QP]
    float4* Rs = geo_s + NG * QP;                                  // [EC][cb][L1p / 4]: c_l R~[e, ch, l], zero padded

    const int tid = threadIdx.x;
    const long long item = blockIdx.x;
    const long long i = item / nblk;
    const int kc0 = (int)(item - i * nblk) * cb;
    const int ncb = (Cpar - kc0 < cb) ? (Cpar - kc0) : cb;

    const int cg = tid / QP, q = tid - cg * QP;
    const bool active = cg < G_;
    int ch[NA];
    bool live[NA];
#pragma unroll
    for (int x = 0; x < NA; ++x) {
        ch[x] = x * G_ + cg;
        live[x] = active && ch[x] < ncb;
    }
    {
        const float4* geo4 = reinterpret_cast<const float4*>(p.geo);
        for (int idx = tid; idx < NG * QP; idx += LR_NT) geo_s[idx] = geo4[idx];
    }
    const int qq = active ? q : 0;
    int roff[NA];  // row of the thread's channels in the staged R~ (float4 units); dead lanes read row 0, never stored
#pragma unroll
    for (int x = 0; x < NA; ++x) roff[x] = live[x] ? ch[x] * (L1p / 4) : 0;
    const float2 z2 = make_float2(0.f, 0.f);
    float2 acc[NA][NF][2];
#pragma unroll
    for (int x = 0; x < NA; ++x)
#pragma unroll
        for (int f = 0; f < NF; ++f) acc[x][f][0] = acc[x][f][1] = z2;

    const bool graph_ok = (*status == 0);
    const long long e_begin = graph_ok ? row_ptr[i] : 0, e_end = graph_ok ? row_ptr[i + 1] : 0;
    __syncthreads();

    for (long long e0 = e_begin; e0 < e_end; e0 += EC) {
        const int ne = (int)((e_end - e0 < EC) ? (e_end - e0) : EC);
        // c_l R~[e, ch, l] of the chunk (the (2l+1)/(4 pi) of the addition theorem folded in), rows padded to float4s
        for (int idx = tid; idx < ne * ncb * L1p; idx += LR_NT) {
            const int el = idx / (ncb * L1p), rem = idx - el * (ncb * L1p);
            const int k = rem / L1p, l = rem - k * L1p;
            float v = 0.f;
            if (l < L1) v = (2.f * l + 1.f) * 0.07957747154594767f * radial[((e0 + el) * (long long)C + perm_par[kc0 + k]) * L1 + l];
            reinterpret_cast<float*>(Rs)[(el * cb + k) * L1p + l] = v;
        }
        if (tid < ne) {
            const long long e = e0 + tid;
            const float ex = edge_vec[3 * e], ey = edge_vec[3 * e + 1], ez = edge_vec[3 * e + 2];
            const float rn = rsqrtf(ex * ex + ey * ey + ez * ez);
            Es[tid] = make_float4(ex * rn, ey * rn, ez * rn, 0.f);
            Ss[tid] = snd[e];
        }
        __syncthreads();

        // the sender grids are fetched one edge ahead: with the degree loop unrolled the kernel waits on these loads
        // (long-scoreboard stalls 4.4 per issue), no longer on the issue slots
        // (measured: odd kernel 15.6 -> 14.3 ms; the even kernel, whose loads the compiler already hoists, 12.2 -> 12.4 ms)
        constexpr bool PF = ODD;
        float4 gn[NA];
        if (PF) {
            const float4* gsrc = reinterpret_cast<const float4*>(G + ((size_t)Ss[0] * Cpar + kc0) * UVp);
#pragma unroll
            for (int x = 0; x < NA; ++x) gn[x] = live[x] ? lr_ldg_stream(gsrc + (size_t)ch[x] * QP + q) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
        for (int el = 0; el < ne; ++el) {
            const float4 ev = Es[el];
            float4 g[NA];
            if (PF) {
#pragma unroll
                for (int x = 0; x < NA; ++x) g[x] = gn[x];
            } else {
                const float4* gsrc = reinterpret_cast<const float4*>(G + ((size_t)Ss[el] * Cpar + kc0) * UVp);
#pragma unroll
                for (int x = 0; x < NA; ++x) g[x] = live[x] ? lr_ldg_stream(gsrc + (size_t)ch[x] * QP + q) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
            if (PF && el + 1 < ne) {
                const float4* gsrc = reinterpret_cast<const float4*>(G + ((size_t)Ss[el + 1] * Cpar + kc0) * UVp);
#pragma unroll
                for (int x = 0; x < NA; ++x) gn[x] = live[x] ? lr_ldg_stream(gsrc + (size_t)ch[x] * QP + q) : make_float4(0.f, 0.f, 0.f, 0.f);
            }

            // E[x] = sum_l (c_l R~[e, ch_x, l]) P_l(t)  (even)  or  sum_l (c_l R~) P'_l(t)  (odd) at the quad's four points,
            // two points per packed operation
            const float4 t4 = lr_dot3(ev.x, ev.y, ev.z, geo_s[qq], geo_s[QP + qq], geo_s[2 * QP + qq]);
            const float2 t[2] = {make_float2(t4.x, t4.y), make_float2(t4.z, t4.w)};
            float2 Ex[NA][2];
#pragma unroll
            for (int x = 0; x < NA; ++x) Ex[x][0] = Ex[x][1] = z2;
            const float4* rrow = Rs + (size_t)el * cb * (L1p / 4);
            const float2 one2 = make_float2(1.f, 1.f);
            float2 pm[2] = {one2, one2}, pc[2] = {t[0], t[1]}, dc[2] = {one2, one2};
#pragma unroll
            for (int l0 = 0; l0 <= LB; l0 += 4) {
                float r[NA][4];
#pragma unroll
                for (int x = 0; x < NA; ++x) {
                    const float4 r4 = rrow[roff[x] + l0 / 4];
                    r[x][0] = r4.x; r[x][1] = r4.y; r[x][2] = r4.z; r[x][3] = r4.w;
                }
#pragma unroll
                for (int dl = 0; dl < 4; ++dl) {
                    const int l = l0 + dl;
                    if (l > LB) break;
                    float2 term[2];
                    if (l == 0) {
                        term[0] = term[1] = ODD ? z2 : one2;  // P_0 = 1, P'_0 = 0
                    } else if (l == 1) {
                        term[0] = ODD ? one2 : t[0];          // P_1 = t, P'_1 = 1
                        term[1] = ODD ? one2 : t[1];
                    } else {
                        const float ca = (2.f * l - 1.f) / l, cb2 = -(l - 1.f) / l, cl = (float)l;
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            const float2 pn = __ffma2_rn(__fmul2_rn(make_float2(ca, ca), t[h]), pc[h],
                                                         __fmul2_rn(make_float2(cb2, cb2), pm[h]));
                            if (ODD) {
                                const float2 dn = __ffma2_rn(t[h], dc[h], __fmul2_rn(make_float2(cl, cl), pc[h]));
                                dc[h] = dn;
                                term[h] = dn;
                            } else {
                                term[h] = pn;
                            }
                            pm[h] = pc[h];
                            pc[h] = pn;
                        }
                    }
#pragma unroll
                    for (int x = 0; x < NA; ++x) {
                        const float2 r2 = make_float2(r[x][dl], r[x][dl]);
                        Ex[x][0] = __ffma2_rn(r2, term[0], Ex[x][0]);
                        Ex[x][1] = __ffma2_rn(r2, term[1], Ex[x][1]);
                    }
                }
            }
            if (!ODD) {
#pragma unroll
                for (int x = 0; x < NA; ++x) {
                    acc[x][0][0] = __ffma2_rn(Ex[x][0], make_float2(g[x].x, g[x].y), acc[x][0][0]);
                    acc[x][0][1] = __ffma2_rn(Ex[x][1], make_float2(g[x].z, g[x].w), acc[x][0][1]);
                }
            } else {
                // X0 += (d_theta E) I,  X1 += -((1/sin) d_phi E) I
                const float4 dth = lr_dot3(ev.x, ev.y, ev.z, geo_s[3 * QP + qq], geo_s[4 * QP + qq], geo_s[5 * QP + qq]);
                const float4 fx = geo_s[6 * QP + qq], fy = geo_s[7 * QP + qq];
                const float4 dph = make_float4(-fmaf(ev.x, fx.x, ev.y * fy.x), -fmaf(ev.x, fx.y, ev.y * fy.y),
                                               -fmaf(ev.x, fx.z, ev.y * fy.z), -fmaf(ev.x, fx.w, ev.y * fy.w));
#pragma unroll
                for (int x = 0; x < NA; ++x) {
                    const float2 g0 = make_float2(g[x].x, g[x].y), g1 = make_float2(g[x].z, g[x].w);
                    const float2 a0 = __fmul2_rn(Ex[x][0], g0), a1 = __fmul2_rn(Ex[x][1], g1);
                    acc[x][0][0] = __ffma2_rn(a0, make_float2(dth.x, dth.y), acc[x][0][0]);
                    acc[x][0][1] = __ffma2_rn(a1, make_float2(dth.z, dth.w), acc[x][0][1]);
                    acc[x][NF - 1][0] = __ffma2_rn(a0, make_float2(dph.x, dph.y), acc[x][NF - 1][0]);
                    acc[x][NF - 1][1] = __ffma2_rn(a1, make_float2(dph.z, dph.w), acc[x][NF - 1][1]);
                }
            }
        }
        __syncthreads();
    }

    float4* sdst = reinterpret_cast<float4*>(S + ((size_t)i * Cpar + kc0) * NF * UVp);
#pragma unroll
    for (int x = 0; x < NA; ++x) {
        if (!live[x]) continue;
#pragma unroll
        for (int f = 0; f < NF; ++f)
            sdst[((size_t)ch[x] * NF + f) * QP + q] =
                make_float4(acc[x][f][0].x, acc[x][f][0].y, acc[x][f][1].x, acc[x][f][1].y);
    }
}

int launch_edge_lr(const Plan* p, bool odd, const float* G, const int64_t* row_ptr, const int64_t* edge_index, int64_t E,
                   const float* edge_vec, const float* edge_radial, const int* perm_par, int Cpar, int C, float* S,
                   int64_t nodes, const int32_t* status, cudaStream_t st)
{
    (void)E;
    if (Cpar <= 0 || nodes <= 0) return CGTP_OK;
    const int QP = p->UVp / 4;
    if (QP > LR_NT || p->lmax >= LR_LMAX) { set_error("edge kernel (l1-dependent radial): grid of lmax=%d too large", p->lmax); return CGTP_ERR_UNSUPPORTED; }
    const int G_ = LR_NT / QP;
    const int NA = 4;
    const int cb_max = NA * G_;
    const int nblk = (Cpar + cb_max - 1) / cb_max;
    int cb = (Cpar + nblk - 1) / nblk;
    cb = std::min(cb_max, (cb + G_ - 1) / G_ * G_);
    // whole in-edge lists in one chunk where they fit: the staging of R~ (two dependent global loads and two barriers
    // per chunk) is exposed, one CTA per SM
    const size_t fixed = (size_t)LR_EC * 16 + LR_EC * 8 + (size_t)(odd ? 8 : 3) * QP * 16;
    const int L1p = round_up(p->LB + 1, 4);
    int EC = LR_EC;
    while (EC > 1 && fixed + (size_t)EC * cb * L1p * 4 > 160 * 1024) EC >>= 1;
    const size_t smem = fixed + (size_t)EC * cb * L1p * 4;
    if (smem > 200 * 1024) { set_error("edge kernel (l1-dependent radial): channel block too large"); return CGTP_ERR_UNSUPPORTED; }
    const int64_t grid = nodes * (int64_t)((Cpar + cb - 1) / cb);
    if (grid > 2147483647LL) { set_error("edge kernel (l1-dependent radial): too many work items"); return CGTP_ERR_UNSUPPORTED; }
    const int nb = (Cpar + cb - 1) / cb;
    LaunchScope scope(odd ? K_EDGE_ODD : K_EDGE_EVEN, st);
    void (*kern)(Plan, const float*, const int64_t*, const int64_t*, const float*, const float*, const int*, int, int, int, int,
                 int, int, float*, const int32_t*) = nullptr;
    switch (p->LB) {
#define CGTP_CASE(B) \
    case B:          \
        kern = odd ? edge_lr_kernel<true, 4, B> : edge_lr_kernel<false, 4, B>; \
        break;
        CGTP_FOR_EACH_BAND(CGTP_CASE)
#undef CGTP_CASE
    }
    if (!kern) { set_error("edge kernel (l1-dependent radial): no kernel for band limit %d", p->LB); return CGTP_ERR_UNSUPPORTED; }
    CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<(unsigned)grid, LR_NT, smem, st>>>(*p, G, row_ptr, edge_index, edge_vec, edge_radial, perm_par, Cpar, C, cb, nb, G_, EC,
                                              S, status);
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

}  // namespace cgtp
