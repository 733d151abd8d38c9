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
constexpr int LR_EC = 8;     // edges per chunk
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

template <bool ODD, int NA>
__global__ void __launch_bounds__(LR_NT, 1) edge_lr_kernel(Plan p, const float* __restrict__ G,
                                                          const int64_t* __restrict__ row_ptr,
                                                          const int64_t* __restrict__ snd,
                                                          const float* __restrict__ edge_vec,
                                                          const float* __restrict__ radial,
                                                          const int* __restrict__ perm_par, int Cpar, int C, int cb,
                                                          int nblk, int G_, float* __restrict__ S,
                                                          const int32_t* __restrict__ status)
{
    constexpr int NF = ODD ? 2 : 1;
    extern __shared__ __align__(16) unsigned char smem_lr[];
    float4* coef = reinterpret_cast<float4*>(smem_lr);             // [LR_LMAX]: (2l-1)/l, -(l-1)/l, (2l+1)/(4 pi), l
    float4* Es = coef + LR_LMAX;                                   // [EC] unit vectors
    long long* Ss = reinterpret_cast<long long*>(Es + LR_EC);      // [EC] senders
    float* Rs = reinterpret_cast<float*>(Ss + LR_EC);              // [EC][cb][L1]

    const int tid = threadIdx.x;
    const int UVp = p.UVp, QP = UVp / 4, lmax = p.lmax, L1 = lmax + 1;
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
    if (tid < LR_LMAX) {
        const float l = (float)(tid > 0 ? tid : 1);
        coef[tid] = make_float4((2.f * l - 1.f) / l, -(l - 1.f) / l, (2.f * tid + 1.f) * 0.07957747154594767f, l);
    }
    // grid geometry of the thread's quad (zero beyond the U*V real points: those columns stay zero)
    const float4* geo4 = reinterpret_cast<const float4*>(p.geo);
    const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
    const float4 gx = active ? geo4[q] : zero4, gy = active ? geo4[QP + q] : zero4, gz = active ? geo4[2 * QP + q] : zero4;
    float4 thx = zero4, thy = zero4, thz = zero4, phx = zero4, phy = zero4;
    if (ODD && active) {
        thx = geo4[3 * QP + q]; thy = geo4[4 * QP + q]; thz = geo4[5 * QP + q];
        phx = geo4[6 * QP + q]; phy = geo4[7 * QP + q];
    }
    const bool pad = 4 * q + 3 >= p.UV;  // quad touches the zero padding of the field
    float4 acc[NA][NF];
#pragma unroll
    for (int x = 0; x < NA; ++x)
#pragma unroll
        for (int f = 0; f < NF; ++f) acc[x][f] = zero4;

    const bool graph_ok = (*status == 0);
    const long long e_begin = graph_ok ? row_ptr[i] : 0, e_end = graph_ok ? row_ptr[i + 1] : 0;
    __syncthreads();

    for (long long e0 = e_begin; e0 < e_end; e0 += LR_EC) {
        const int ne = (int)((e_end - e0 < LR_EC) ? (e_end - e0) : LR_EC);
        for (int idx = tid; idx < ne * ncb * L1; idx += LR_NT) {
            const int el = idx / (ncb * L1), rem = idx - el * (ncb * L1);
            const int k = rem / L1, l = rem - k * L1;
            Rs[(el * cb + k) * L1 + l] = radial[((e0 + el) * (long long)C + perm_par[kc0 + k]) * L1 + l];
        }
        if (tid < ne) {
            const long long e = e0 + tid;
            const float ex = edge_vec[3 * e], ey = edge_vec[3 * e + 1], ez = edge_vec[3 * e + 2];
            const float rn = rsqrtf(ex * ex + ey * ey + ez * ez);
            Es[tid] = make_float4(ex * rn, ey * rn, ez * rn, 0.f);
            Ss[tid] = snd[e];
        }
        __syncthreads();

        for (int el = 0; el < ne; ++el) {
            const float4 ev = Es[el];
            const float4* gsrc = reinterpret_cast<const float4*>(G + ((size_t)Ss[el] * Cpar + kc0) * UVp);
            float4 g[NA];
#pragma unroll
            for (int x = 0; x < NA; ++x) g[x] = live[x] ? lr_ldg_stream(gsrc + (size_t)ch[x] * QP + q) : zero4;

            // E[x] = sum_l R~[e, ch_x, l] c_l P_l(t)   (even)   or   sum_l R~ c_l P'_l(t)   (odd), at the quad's points
            const float4 t = lr_dot3(ev.x, ev.y, ev.z, gx, gy, gz);
            float4 Ex[NA];
#pragma unroll
            for (int x = 0; x < NA; ++x) Ex[x] = zero4;
            const float* rrow = Rs + (size_t)el * cb * L1;
            float4 pm = make_float4(1.f, 1.f, 1.f, 1.f), pc = t, dc = make_float4(1.f, 1.f, 1.f, 1.f);
            if (!ODD) {
                const float c0 = coef[0].z;
#pragma unroll
                for (int x = 0; x < NA; ++x) {
                    const float r = live[x] ? rrow[ch[x] * L1] : 0.f;
                    lr_axpy(Ex[x], r * c0, pm);
                }
            }
            if (lmax >= 1) {
                const float c1 = coef[1].z;
                const float4 term = ODD ? dc : pc;  // P'_1 = 1, P_1 = t
#pragma unroll
                for (int x = 0; x < NA; ++x) {
                    const float r = live[x] ? rrow[ch[x] * L1 + 1] : 0.f;
                    lr_axpy(Ex[x], r * c1, term);
                }
            }
            for (int l = 2; l <= lmax; ++l) {
                const float4 c = coef[l];
                float4 pn, dn = zero4;
                pn.x = fmaf(c.x * t.x, pc.x, c.y * pm.x); pn.y = fmaf(c.x * t.y, pc.y, c.y * pm.y);
                pn.z = fmaf(c.x * t.z, pc.z, c.y * pm.z); pn.w = fmaf(c.x * t.w, pc.w, c.y * pm.w);
                if (ODD) {
                    dn.x = fmaf(t.x, dc.x, c.w * pc.x); dn.y = fmaf(t.y, dc.y, c.w * pc.y);
                    dn.z = fmaf(t.z, dc.z, c.w * pc.z); dn.w = fmaf(t.w, dc.w, c.w * pc.w);
                }
                const float4 term = ODD ? dn : pn;
#pragma unroll
                for (int x = 0; x < NA; ++x) {
                    const float r = live[x] ? rrow[ch[x] * L1 + l] : 0.f;
                    lr_axpy(Ex[x], r * c.z, term);
                }
                pm = pc; pc = pn; dc = dn;
            }
            if (!ODD) {
#pragma unroll
                for (int x = 0; x < NA; ++x) lr_fma4(acc[x][0], Ex[x], g[x]);
            } else {
                // X0 += (d_theta E) I,  X1 += -((1/sin) d_phi E) I
                const float4 dth = lr_dot3(ev.x, ev.y, ev.z, thx, thy, thz);
                const float4 dph = make_float4(-fmaf(ev.x, phx.x, ev.y * phy.x), -fmaf(ev.x, phx.y, ev.y * phy.y),
                                               -fmaf(ev.x, phx.z, ev.y * phy.z), -fmaf(ev.x, phx.w, ev.y * phy.w));
#pragma unroll
                for (int x = 0; x < NA; ++x) {
                    const float4 a = make_float4(Ex[x].x * dth.x, Ex[x].y * dth.y, Ex[x].z * dth.z, Ex[x].w * dth.w);
                    const float4 b = make_float4(Ex[x].x * dph.x, Ex[x].y * dph.y, Ex[x].z * dph.z, Ex[x].w * dph.w);
                    lr_fma4(acc[x][0], a, g[x]);
                    lr_fma4(acc[x][NF - 1], b, g[x]);
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
        for (int f = 0; f < NF; ++f) {
            float4 v = acc[x][f];
            if (pad) {  // the even field K(t) does not vanish at the padded points (their geometry is zero, t = 0)
                const int b = 4 * q;
                if (b + 0 >= p.UV) v.x = 0.f;
                if (b + 1 >= p.UV) v.y = 0.f;
                if (b + 2 >= p.UV) v.z = 0.f;
                if (b + 3 >= p.UV) v.w = 0.f;
            }
            sdst[((size_t)ch[x] * NF + f) * QP + q] = v;
        }
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
    const int NA = odd ? 2 : 4;
    const int cb_max = NA * G_;
    const int nblk = (Cpar + cb_max - 1) / cb_max;
    int cb = (Cpar + nblk - 1) / nblk;
    cb = std::min(cb_max, (cb + G_ - 1) / G_ * G_);
    const int L1 = p->lmax + 1;
    const size_t smem = (size_t)LR_LMAX * 16 + LR_EC * 16 + LR_EC * 8 + (size_t)LR_EC * cb * L1 * 4;
    if (smem > 200 * 1024) { set_error("edge kernel (l1-dependent radial): channel block too large"); return CGTP_ERR_UNSUPPORTED; }
    const int64_t grid = nodes * (int64_t)((Cpar + cb - 1) / cb);
    if (grid > 2147483647LL) { set_error("edge kernel (l1-dependent radial): too many work items"); return CGTP_ERR_UNSUPPORTED; }
    const int nb = (Cpar + cb - 1) / cb;
    LaunchScope scope(odd ? K_EDGE_ODD : K_EDGE_EVEN, st);
    if (odd) {
        auto kern = edge_lr_kernel<true, 2>;
        CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kern<<<(unsigned)grid, LR_NT, smem, st>>>(*p, G, row_ptr, edge_index, edge_vec, edge_radial, perm_par, Cpar, C, cb, nb,
                                                  G_, S, status);
    } else {
        auto kern = edge_lr_kernel<false, 4>;
        CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kern<<<(unsigned)grid, LR_NT, smem, st>>>(*p, G, row_ptr, edge_index, edge_vec, edge_radial, perm_par, Cpar, C, cb, nb,
                                                  G_, S, status);
    }
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

}  // namespace cgtp
