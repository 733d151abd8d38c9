// message.cu -- message-passing kernels (rows M0, M2, M3, M4, M5 of SURVEY.md 8(a); Sec. VII C).
//
// Data flow (paper-faithful "gather sender grids", PAPER.md:404-:415):
//   M2  node synthesis   H[j,c,:] -> grid fields G[j,c,(u,v)]              (Eq.(49),(51)), once per node
//   M3+M4 edge kernel    S[i,c,(u,v)] = sum_{e -> i} E_e(u,v) (x) G[send(e),c,(u,v)]  (Eq.(48),(50),(52),(57))
//                        one CTA per (receiver, channel block); sender grids are streamed from HBM with
//                        128-bit loads; the sum runs in registers in edge order: deterministic,
//                        no floating-point atomics.
//   M5  analysis         T[i,c,lm] from S, once per receiver by linearity  (Eq.(53),(54))
//
// Edge factor with an l1-shared radial function (R12): E_e(Omega) = R~[e,c] K_e(Omega),
//   K_e(Omega) = sum_{l<=lmax} (2l+1)/(4 pi) P_l(r_e . Omega)     (addition theorem)
// and for the odd channels its surface gradient in the (theta_hat, phi_hat) frame:
//   d_theta K_e = k'(t) (r_e . theta_hat),  (1/sin theta) d_phi K_e = k'(t) (r_e . phi_hat),  t = r_e . Omega.
#include <mutex>

#include "sht.cuh"

namespace cgtp {

// =============================================================================================
// M0: segmentation
// =============================================================================================
__global__ void segments_kernel(const int64_t* __restrict__ edge_index, long long E, long long nodes,
                                long long n_send, int64_t* __restrict__ row_ptr, int32_t* __restrict__ status)
{
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e > E) return;
    const int64_t* snd = edge_index;
    const int64_t* rcv = edge_index + E;
    long long r_prev = (e == 0) ? -1 : rcv[e - 1];
    long long r = (e == E) ? nodes : rcv[e];
    bool bad = false;
    if (e < E) {
        const long long s = snd[e];
        if (r < 0 || r >= nodes || s < 0 || s >= n_send) bad = true;
    }
    if (e > 0 && (r_prev < 0 || r_prev >= nodes)) bad = true;
    if (r < r_prev) bad = true;
    if (bad) {
        atomicOr(status, CGTP_ERR_GRAPH);  // integer flag, not a floating-point reduction
        return;
    }
    // rows r_prev+1 .. r start at edge e
    for (long long i = r_prev + 1; i <= r; ++i) row_ptr[i] = e;
}

__global__ void set_status_kernel(int32_t* status, int32_t v) { *status = v; }

int launch_segments(const int64_t* edge_index, int64_t E, int64_t nodes, int64_t n_send, int64_t* row_ptr,
                    int32_t* status, cudaStream_t st)
{
    {
        LaunchScope scope(K_MISC, st);
        set_status_kernel<<<1, 1, 0, st>>>(status, 0);
        CGTP_CUDA_CHECK(cudaGetLastError());
    }
    const int NT = 256;
    int64_t grid = (E + 1 + NT - 1) / NT;
    LaunchScope scope(K_SEGMENTS, st);
    segments_kernel<<<(unsigned)grid, NT, 0, st>>>(edge_index, (long long)E, (long long)nodes, (long long)n_send, row_ptr,
                                                    status);
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

// =============================================================================================
// M2: node synthesis
// =============================================================================================
struct SynthSmem {
    int bar, tab0, tab1, qc, qs, hs, f, g, total;
    int tab_bytes, q_bytes;
};

static SynthSmem synth_smem_layout(const Plan* p, int NC)
{
    SynthSmem s;
    const int M = 2 * p->LB + 1;
    const int J = (NC * p->U) | 1;  // odd row stride: rows of different m fall into different banks
    const int nf = 1;
    s.tab_bytes = p->Uh * p->NTRI * 4;
    s.q_bytes = p->Vh * p->QSTR * 4;
    int off = 0;
    s.bar = off; off += 16;
    s.tab0 = off; off += s.tab_bytes;
    s.tab1 = off;
    s.qc = off; off += s.q_bytes;
    s.qs = off; off += s.q_bytes;
    s.hs = off; off += NC * p->L2p * 4;
    s.f = off; off += round_up(nf * M * J, 4) * 4;
    s.g = off; off += NC * nf * p->UVp * 4;
    s.total = off;
    return s;
}

template <int LB>
__global__ void __launch_bounds__(256) node_synth_kernel(Plan p, SynthSmem lay, const float* __restrict__ H,
                                                        float* __restrict__ G, long long ncols, int NC)
{
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int M = 2 * LB + 1;
    constexpr int NF = 1;
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + lay.bar);
    float* tab0 = reinterpret_cast<float*>(smem + lay.tab0);
    float* qc = reinterpret_cast<float*>(smem + lay.qc);
    float* qs = reinterpret_cast<float*>(smem + lay.qs);
    float* hs = reinterpret_cast<float*>(smem + lay.hs);
    float* F = reinterpret_cast<float*>(smem + lay.f);
    float* Gs = reinterpret_cast<float*>(smem + lay.g);

    const long long col0 = (long long)blockIdx.x * NC;
    const int nc = (int)((ncols - col0 < NC) ? (ncols - col0) : NC);
    const int J = (NC * p.U) | 1;  // odd row stride (matches the host layout)
    const int hbytes = nc * p.L2p * 4;

    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncthreads();
    pdl_launch_dependents();  // programmatic dependent launch, common.cuh
    if (threadIdx.x == 0) {
        const uint32_t total = lay.tab_bytes + 2 * lay.q_bytes + hbytes;
        mbar_arrive_expect_tx(bar, total);
        tma_load_span(tab0, p.PT, lay.tab_bytes, bar);  // the plan's tables: independent of the predecessor
        tma_load_span(qc, p.QC, lay.q_bytes, bar);
        tma_load_span(qs, p.QS, lay.q_bytes, bar);
        pdl_wait();  // H is the predecessor's output; G is written only after it has arrived
        tma_load_span(hs, H + col0 * p.L2p, hbytes, bar);
    }
#pragma unroll
    for (int i = 0; i < NF; ++i) zero_high_rows<LB>(F + (size_t)i * M * J, p.lmax, J);
    // zero the padding of every grid field so the edge kernel can stream whole float4s
    if (p.UVp > p.UV) {
        const int pad = p.UVp - p.UV;
        for (int idx = threadIdx.x; idx < nc * NF * pad; idx += blockDim.x) {
            const int f = idx / pad, q = idx - f * pad;
            Gs[(size_t)f * p.UVp + p.UV + q] = 0.f;
        }
    }
    mbar_wait(bar, 0);

    {
        const LegDst dst[1][2] = {{{F, 1.f}, {nullptr, 0.f}}};
        legendre_synthesis<LB, false, 1, 4>(tab0, nullptr, hs, 0, p.L2p, dst, nc, p.lmax, p.U, p.Uh, p.NTRI, J);
    }
    __syncthreads();

    const int rows = nc * p.U;
    for (int item = threadIdx.x; item < NF * rows; item += blockDim.x) {
        const int f = item / rows;
        const int j = item - f * rows;
        const int col = j / p.U, u = j - col * p.U;
        float* grow = Gs + ((size_t)col * NF + f) * p.UVp + u * p.V;
        dft_forward_row<LB>(F + (size_t)f * M * J, J, j, grow, qc, qs, p.V, p.Vh);
    }
    __syncthreads();

    // coalesced 128-bit store of the CTA's contiguous block of grid fields
    const int n4 = nc * NF * p.UVp / 4;
    float4* dst4 = reinterpret_cast<float4*>(G + col0 * NF * p.UVp);
    const float4* src4 = reinterpret_cast<const float4*>(Gs);
    for (int i = threadIdx.x; i < n4; i += blockDim.x) dst4[i] = src4[i];
}

template <int LB>
static int launch_node_synth_t(const Plan* p, Kind kind, const float* H, float* G, int64_t ncols, cudaStream_t st)
{
    const int M = 2 * p->LB + 1;
    const int nf = 1;
    SynthSmem fixed = synth_smem_layout(p, 0);
    const int percol = p->L2p * 4 + nf * M * p->U * 4 + nf * p->UVp * 4;
    // 45 KB per CTA -> four or five CTAs per SM, so that the load / compute / store phases of different CTAs overlap
    // (measured on configs[2] / configs[4]: 64 -> 52 us and 1.08 -> 0.85 ms against a 100 KB budget)
    int budget = 45 * 1024;
    int NC = (budget - fixed.total - 64) / percol;
    if (NC < 4) {
        budget = 220 * 1024;
        NC = (budget - fixed.total - 64) / percol;
    }
    if (NC < 1) { set_error("node synthesis: shared memory too small for lmax=%d", p->lmax); return CGTP_ERR_UNSUPPORTED; }
    if (NC > 128) NC = 128;
    if ((int64_t)NC > ncols) NC = (int)ncols;
    SynthSmem lay = synth_smem_layout(p, NC);
    auto kern = node_synth_kernel<LB>;
    CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, lay.total));
    int64_t grid = (ncols + NC - 1) / NC;
    LaunchScope scope(kind, st);
    CGTP_CUDA_CHECK(launch_pdl(kern, (unsigned)grid, 256u, (size_t)lay.total, st, *p, lay, H, G, (long long)ncols, NC));
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

int launch_node_synth(const Plan* p, bool odd, const float* H, float* G, int64_t ncols, cudaStream_t st)
{
    if (ncols <= 0) return CGTP_OK;
    switch (p->LB) {
#define CGTP_CASE(B) \
    case B:          \
        return launch_node_synth_t<B>(p, odd ? K_NODE_SYNTH_ODD : K_NODE_SYNTH_EVEN, H, G, ncols, st);
        CGTP_FOR_EACH_BAND(CGTP_CASE)
#undef CGTP_CASE
    }
    set_error("node synthesis: no kernel for band limit %d", p->LB);
    return CGTP_ERR_UNSUPPORTED;
}

// =============================================================================================
// M3 + M4: edge factor, gather, product, segmented sum
// =============================================================================================
constexpr int EDGE_NT = 256;  // threads per CTA
constexpr int EDGE_NI = 8;    // float4 accumulators per thread
constexpr int EDGE_EC = 8;    // edges per geometry chunk

__device__ __forceinline__ float4 ldg_stream(const float4* p)
{
    float4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w)
                 : "l"(p));
    return r;
}

// G   : [nodes][Cpar][UVp] (value field, both parities)
// S   : even [nodes][Cpar][UVp]          odd [nodes][Cpar][2][UVp] = (X0, X1) of the by-parts pairing
// grid: (channel blocks, receivers)
template <bool ODD>
__global__ void __launch_bounds__(EDGE_NT) edge_kernel(Plan p, const float* __restrict__ G,
                                                      const int64_t* __restrict__ row_ptr,
                                                      const int64_t* __restrict__ snd,
                                                      const float* __restrict__ edge_vec,
                                                      const float* __restrict__ edge_radial,
                                                      const int* __restrict__ perm_par, int Cpar, int C, int cb,
                                                      float* __restrict__ S, const int32_t* __restrict__ status)
{
    constexpr int NF = ODD ? 2 : 1;
    extern __shared__ __align__(16) unsigned char smem_e[];
    const int UVp = p.UVp, QP = UVp / 4;
    float* Kbuf = reinterpret_cast<float*>(smem_e);                 // [EC][NF][UVp]
    float* Rbuf = Kbuf + (size_t)EDGE_EC * NF * UVp;                // [EC][cb]
    long long* Sbuf = reinterpret_cast<long long*>(Rbuf + round_up(EDGE_EC * cb, 4));  // [EC]

    const long long i = blockIdx.y;
    const int kc0 = blockIdx.x * cb;
    const int ncb = (Cpar - kc0 < cb) ? (Cpar - kc0) : cb;
    const int n4 = ncb * QP;  // float4 accumulators of this block

    // ownership: accumulator a of this thread is float4 index f = tid + a*NT -> (channel kc, quad q)
    int kcl[EDGE_NI], qd[EDGE_NI];
    float4 acc[EDGE_NI][NF];
#pragma unroll
    for (int a = 0; a < EDGE_NI; ++a) {
        const int f = threadIdx.x + a * EDGE_NT;
        kcl[a] = (f < n4) ? f / QP : -1;
        qd[a] = (f < n4) ? f - kcl[a] * QP : 0;
#pragma unroll
        for (int x = 0; x < NF; ++x) acc[a][x] = make_float4(0.f, 0.f, 0.f, 0.f);
    }

    const bool graph_ok = (*status == 0);
    const long long e_begin = graph_ok ? row_ptr[i] : 0;
    const long long e_end = graph_ok ? row_ptr[i + 1] : 0;
    const float inv4pi = 0.07957747154594767f;

    for (long long e0 = e_begin; e0 < e_end; e0 += EDGE_EC) {
        const int ne = (int)((e_end - e0 < EDGE_EC) ? (e_end - e0) : EDGE_EC);
        // ---- M3: edge fields of the chunk on the grid
        for (int idx = threadIdx.x; idx < ne * UVp; idx += EDGE_NT) {
            const int el = idx / UVp, q = idx - el * UVp;
            const long long e = e0 + el;
            float k0 = 0.f, k1 = 0.f;
            if (q < p.UV) {
                float ex = edge_vec[3 * e], ey = edge_vec[3 * e + 1], ez = edge_vec[3 * e + 2];
                const float rn = rsqrtf(ex * ex + ey * ey + ez * ez);
                ex *= rn; ey *= rn; ez *= rn;
                const float t = ex * p.geo[q] + ey * p.geo[UVp + q] + ez * p.geo[2 * UVp + q];
                // Legendre recurrences: P_l(t), P'_l(t) = t P'_{l-1} + l P_{l-1}
                float pm = 1.f, pc = t, dc = 1.f;
                float ks = inv4pi, kd = 0.f;
                if (p.lmax >= 1) { ks += 3.f * inv4pi * pc; kd += 3.f * inv4pi * dc; }
                for (int l = 2; l <= p.lmax; ++l) {
                    const float pn = ((2 * l - 1) * t * pc - (l - 1) * pm) / l;
                    const float dn = fmaf(t, dc, l * pc);
                    const float c = (2 * l + 1) * inv4pi;
                    ks = fmaf(c, pn, ks);
                    kd = fmaf(c, dn, kd);
                    pm = pc; pc = pn; dc = dn;
                }
                if (!ODD) {
                    k0 = ks;
                } else {
                    const float dth = ex * p.geo[3 * UVp + q] + ey * p.geo[4 * UVp + q] + ez * p.geo[5 * UVp + q];
                    const float dph = ex * p.geo[6 * UVp + q] + ey * p.geo[7 * UVp + q];
                    k0 = kd * dth;
                    k1 = -(kd * dph);
                }
            }
            Kbuf[((size_t)el * NF) * UVp + q] = k0;
            if (ODD) Kbuf[((size_t)el * NF + 1) * UVp + q] = k1;
        }
        for (int idx = threadIdx.x; idx < ne * ncb; idx += EDGE_NT) {
            const int el = idx / ncb, k = idx - el * ncb;
            Rbuf[el * cb + k] = edge_radial[(e0 + el) * C + perm_par[kc0 + k]];
        }
        if (threadIdx.x < ne) Sbuf[threadIdx.x] = snd[e0 + threadIdx.x];
        __syncthreads();

        // ---- M4: gather the sender's grid fields, multiply, accumulate (fixed edge order)
        for (int el = 0; el < ne; ++el) {
            const float4* gsrc = reinterpret_cast<const float4*>(G + ((size_t)Sbuf[el] * Cpar + kc0) * UVp);
            const float4* k4 = reinterpret_cast<const float4*>(Kbuf + (size_t)el * NF * UVp);
            float4 g0[EDGE_NI];
#pragma unroll
            for (int a = 0; a < EDGE_NI; ++a)
                if (kcl[a] >= 0) g0[a] = ldg_stream(gsrc + (size_t)kcl[a] * QP + qd[a]);
#pragma unroll
            for (int a = 0; a < EDGE_NI; ++a) {
                if (kcl[a] >= 0) {
                    const float r = Rbuf[el * cb + kcl[a]];
#pragma unroll
                    for (int x = 0; x < NF; ++x) {
                        // even: K_e; odd: (d_theta K_e, -(1/sin) d_phi K_e) against the sender's value field
                        const float4 k = k4[x * QP + qd[a]];
                        acc[a][x].x = fmaf(r * k.x, g0[a].x, acc[a][x].x);
                        acc[a][x].y = fmaf(r * k.y, g0[a].y, acc[a][x].y);
                        acc[a][x].z = fmaf(r * k.z, g0[a].z, acc[a][x].z);
                        acc[a][x].w = fmaf(r * k.w, g0[a].w, acc[a][x].w);
                    }
                }
            }
        }
        __syncthreads();
    }

    float4* sdst = reinterpret_cast<float4*>(S + ((size_t)i * Cpar + kc0) * NF * UVp);
#pragma unroll
    for (int a = 0; a < EDGE_NI; ++a)
        if (kcl[a] >= 0) {
#pragma unroll
            for (int x = 0; x < NF; ++x) sdst[((size_t)kcl[a] * NF + x) * QP + qd[a]] = acc[a][x];
        }
}

int launch_edge(const Plan* p, bool odd, const float* G, const int64_t* row_ptr, const int64_t* edge_index, int64_t E,
                const float* edge_vec, const float* edge_radial, const int* perm_par, int Cpar, int C, float* S,
                int64_t nodes, const int32_t* status, cudaStream_t st)
{
    if (Cpar <= 0 || nodes <= 0) return CGTP_OK;
    if (!(kernel_path() & PATH_GENERIC_EDGE)) {
        bool handled = false;
        const int rc = launch_edge_ring(p, odd, G, row_ptr, edge_index, E, edge_vec, edge_radial, perm_par, Cpar, C, S,
                                        nodes, status, st, &handled);
        if (rc != CGTP_OK || handled) return rc;
    }
    const int QP = p->UVp / 4;
    int cbmax = EDGE_NI * EDGE_NT / QP;
    if (cbmax < 1) { set_error("edge kernel: grid of lmax=%d too large for the accumulator tile", p->lmax); return CGTP_ERR_UNSUPPORTED; }
    int nblk = (Cpar + cbmax - 1) / cbmax;
    int cb = (Cpar + nblk - 1) / nblk;
    const int nf = odd ? 2 : 1;
    size_t smem = (size_t)EDGE_EC * nf * p->UVp * 4 + (size_t)round_up(EDGE_EC * cb, 4) * 4 + EDGE_EC * 8;
    dim3 grid(nblk, 1, 1);
    LaunchScope scope(odd ? K_EDGE_ODD : K_EDGE_EVEN, st);
    // receivers go on grid.y (max 65535) in slabs
    for (int64_t n0 = 0; n0 < nodes; n0 += 65535) {
        int64_t nn = nodes - n0 < 65535 ? nodes - n0 : 65535;
        grid.y = (unsigned)nn;
        if (odd) {
            CGTP_CUDA_CHECK(cudaFuncSetAttribute(edge_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            edge_kernel<true><<<grid, EDGE_NT, smem, st>>>(*p, G, row_ptr + n0, edge_index, edge_vec, edge_radial, perm_par,
                                                          Cpar, C, cb, S + (size_t)n0 * Cpar * 2 * p->UVp, status);
        } else {
            CGTP_CUDA_CHECK(cudaFuncSetAttribute(edge_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            edge_kernel<false><<<grid, EDGE_NT, smem, st>>>(*p, G, row_ptr + n0, edge_index, edge_vec, edge_radial, perm_par,
                                                           Cpar, C, cb, S + (size_t)n0 * Cpar * p->UVp, status);
        }
        CGTP_CUDA_CHECK(cudaGetLastError());
    }
    (void)E;
    return CGTP_OK;
}

// =============================================================================================
// M5: analysis of the pooled grids
// =============================================================================================
struct AnaSmem {
    int bar, wp, qc, qs, wv, ss, t, total;
    int tab_bytes, q_bytes, wv_bytes;
};

static AnaSmem ana_smem_layout(const Plan* p, bool odd, int NC)
{
    AnaSmem s;
    const int M = 2 * p->LB + 1;
    const int J = (NC * p->U) | 1;  // odd row stride: rows of different m fall into different banks
    const int nf = odd ? 2 : 1;     // odd channels: the field pair (X0, X1) and the table pair (WD, WS)
    s.tab_bytes = p->Uh * p->NTRI * 4;
    s.q_bytes = p->Vh * p->QSTR * 4;
    s.wv_bytes = round_up(p->Vh, 4) * 4;
    int off = 0;
    s.bar = off; off += 16;
    s.wp = off; off += nf * s.tab_bytes;
    s.qc = s.qs = s.wv = off;  // the azimuthal tables are a kernel parameter (QParam)
    s.ss = off; off += NC * nf * p->UVp * 4;
    s.t = off; off += nf * round_up(M * J, 4) * 4;
    s.total = off;
    return s;
}

template <int LB, bool ODD>
__global__ void __launch_bounds__(256) analysis_kernel(Plan p, AnaSmem lay, const __grid_constant__ QParam<LB> qp,
                                                      const float* __restrict__ S, float* __restrict__ T, long long ncols,
                                                      int NC)
{
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int M = 2 * LB + 1;
    constexpr int NF = ODD ? 2 : 1;
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + lay.bar);
    float* wp = reinterpret_cast<float*>(smem + lay.wp);
    float* Ss = reinterpret_cast<float*>(smem + lay.ss);
    float* Tm = reinterpret_cast<float*>(smem + lay.t);

    const long long col0 = (long long)blockIdx.x * NC;
    const int nc = (int)((ncols - col0 < NC) ? (ncols - col0) : NC);
    const int J = (NC * p.U) | 1;  // odd row stride (matches the host layout)
    const int MJ = round_up(M * J, 4);
    const int sbytes = nc * NF * p.UVp * 4;

    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncthreads();
    pdl_launch_dependents();  // programmatic dependent launch, common.cuh
    if (threadIdx.x == 0) {
        const uint32_t total = NF * lay.tab_bytes + sbytes;
        mbar_arrive_expect_tx(bar, total);
        if (!ODD) {
            tma_load_span(wp, p.WP, lay.tab_bytes, bar);  // the plan's tables: independent of the predecessor
        } else {
            tma_load_span(wp, p.WD, lay.tab_bytes, bar);
            tma_load_span(wp + lay.tab_bytes / 4, p.WS, lay.tab_bytes, bar);
        }
        pdl_wait();  // S is the predecessor's output; T is written only after it has arrived
        tma_load_span(Ss, S + col0 * NF * p.UVp, sbytes, bar);
    }
    mbar_wait(bar, 0);

    const int rows = nc * p.U;
    for (int item = threadIdx.x; item < NF * rows; item += blockDim.x) {
        const int f = item / rows, j = item - f * rows;
        const int col = j / p.U, u = j - col * p.U;
        dft_inverse_row_p<LB>(Ss + ((size_t)col * NF + f) * p.UVp + u * p.V, Tm + (size_t)f * MJ, J, j, qp, p.V, p.Vh);
    }
    __syncthreads();
    if (!ODD)
        legendre_analysis<LB>(Tm, nullptr, wp, T + col0 * p.Lo2p, p.Lo2p, nc, p.lmax_out, p.U, p.Uh, p.NTRI, J);
    else
        legendre_analysis_curl<LB>(Tm, Tm + MJ, wp, wp + lay.tab_bytes / 4, T + col0 * p.Lo2p, p.Lo2p, nc, p.lmax_out, p.U,
                                   p.Uh, p.NTRI, J);
}

template <int LB, bool ODD>
static int launch_analysis_t(const Plan* p, const float* S, float* T, int64_t ncols, cudaStream_t st)
{
    const int M = 2 * p->LB + 1;
    const int nf = ODD ? 2 : 1;
    AnaSmem fixed = ana_smem_layout(p, ODD, 0);
    const int percol = nf * (p->UVp * 4 + M * p->U * 4);
    int budget = 45 * 1024;  // as node synthesis: several small CTAs per SM overlap their phases (0.80 -> 0.67 ms, configs[4])
    int NC = (budget - fixed.total - 64) / percol;
    if (NC < 4) {
        budget = 220 * 1024;
        NC = (budget - fixed.total - 64) / percol;
    }
    if (NC < 1) { set_error("analysis: shared memory too small for lmax=%d", p->lmax); return CGTP_ERR_UNSUPPORTED; }
    if (NC > 128) NC = 128;
    if ((int64_t)NC > ncols) NC = (int)ncols;
    AnaSmem lay = ana_smem_layout(p, ODD, NC);
    auto kern = analysis_kernel<LB, ODD>;
    CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, lay.total));
    int64_t grid = (ncols + NC - 1) / NC;
    LaunchScope scope(ODD ? K_ANALYSIS_ODD : K_ANALYSIS_EVEN, st);
    QParam<LB> qp;
    fill_qparam<LB>(p, qp);
    CGTP_CUDA_CHECK(launch_pdl(kern, (unsigned)grid, 256u, (size_t)lay.total, st, *p, lay, qp, S, T, (long long)ncols, NC));
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

int launch_analysis(const Plan* p, bool odd, const float* S, float* T, int64_t ncols, cudaStream_t st)
{
    if (ncols <= 0) return CGTP_OK;
    switch (p->LB) {
#define CGTP_CASE(B) \
    case B:          \
        return odd ? launch_analysis_t<B, true>(p, S, T, ncols, st) : launch_analysis_t<B, false>(p, S, T, ncols, st);
        CGTP_FOR_EACH_BAND(CGTP_CASE)
#undef CGTP_CASE
    }
    set_error("analysis: no kernel for band limit %d", p->LB);
    return CGTP_ERR_UNSUPPORTED;
}

}  // namespace cgtp
