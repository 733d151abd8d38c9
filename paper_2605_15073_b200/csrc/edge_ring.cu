// edge_ring.cu -- rows M3 + M4 of SURVEY.md 8(a) (edge factor, gather, product / surface-curl pairing,
// neighbour sum; Eq.(48),(50),(52) :402-:415, Eq.(57) :443) as a persistent, warp-specialised
// streaming kernel:
//   * one CTA per SM loops over (receiver, channel block) items; a producer warp walks the receiver's
//     in-edges and streams the sender's grid block from HBM into a shared-memory ring with TMA bulk
//     copies (cp.async.bulk + mbarrier complete_tx), one stage = one (edge, channel sub-block) span,
//     contiguous and 16-byte aligned in the G layout of message.cu;
//   * eight consumer warps evaluate the channel-independent edge field K_e on the grid (Legendre
//     recurrence in r_e . Omega, chunks of edges), multiply it and R~[e,c] with the staged sender grid
//     and accumulate in registers in input edge order -- deterministic, no floating-point atomics;
//   * the ring keeps tens of KB per SM in flight independent of occupancy, which is what an
//     HBM-latency-bound gather needs; S is written once per receiver with 128-bit stores.
// The arithmetic per grid point is identical to edge_kernel in message.cu (kept as the fallback).
#include <algorithm>

#include "sht.cuh"

namespace cgtp {

constexpr int ER_CONS = 512;            // consumer threads
constexpr int ER_NT = ER_CONS + 32;     // + producer warp
// float4 accumulators per thread per sub-block (template parameter NA): 2 for the odd kernel (two fields per channel),
// 4 for the even one, so that a ring stage carries the same ~31 KB and a thread has the same number of independent
// load -> multiply -> accumulate chains per mbarrier hand-over in both (with 2 the even kernel was latency-bound at
// 5.6 TB/s against 7.1 TB/s for the odd one)
constexpr int ER_MAXST = 16;            // ring stages (upper bound)
constexpr int ER_LMAX = 24;             // recurrence coefficient table length

struct EdgeRingArgs {
    Plan p;
    const float* G;
    const int64_t* row_ptr;
    const int64_t* snd;
    const float* edge_vec;
    const float* edge_radial;
    const int* perm_par;
    float* S;
    const int32_t* status;
    long long nodes;
    int Cpar, C;
    int cb;     // channels per CTA block
    int nblk;   // channel blocks
    int cs;     // channels per sub-block (one ring stage)
    int G_;     // channel groups per sub-block pass: 512 / QP
    int EC;     // edges per geometry chunk
    int NST;    // ring stages
    int geo_smem;  // 1: grid geometry staged in shared memory
    int stage_bytes, k_bytes, r_bytes, geo_bytes;
};

__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void consumer_sync() { asm volatile("bar.sync 1, %0;" ::"n"(ER_CONS) : "memory"); }

__device__ __forceinline__ float2 lo2(const float4& v) { return make_float2(v.x, v.y); }
__device__ __forceinline__ float2 hi2(const float4& v) { return make_float2(v.z, v.w); }

// Thread <-> accumulator mapping (QP <= 512 float4 quads per grid field, true for every band limit the
// library compiles): thread = (channel group cg, quad q0), accumulator x of a sub-block = channel
// x*G + cg at quad q0, so the edge field at q0 stays in registers for every channel of the edge.
template <bool ODD, int NSBT, int NA>
__global__ void __launch_bounds__(ER_NT, 1) edge_ring_kernel(EdgeRingArgs a)
{
    constexpr int NF = ODD ? 2 : 1;
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);   // [ER_MAXST]
    uint64_t* empty = full + ER_MAXST;                    // [ER_MAXST]
    float* coef = reinterpret_cast<float*>(smem + 256);   // [3][ER_LMAX]: (2l-1)/l, (l-1)/l, (2l+1)/(4 pi)
    float* geo_s = coef + 3 * ER_LMAX;
    float* Kbuf = reinterpret_cast<float*>(smem + 256 + 3 * ER_LMAX * 4 + a.geo_bytes);  // [EC][NF][UVp]
    float* Rbuf = Kbuf + a.k_bytes / 4;                                                   // [EC][cb]
    unsigned char* ring = reinterpret_cast<unsigned char*>(Rbuf) + a.r_bytes;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int UVp = a.p.UVp, QP = UVp / 4;
    const int NST = a.NST, cs = a.cs, cb = a.cb, nblk = a.nblk, Cpar = a.Cpar;

    if (tid == 0) {
        for (int s = 0; s < NST; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], ER_CONS / 32);
        }
        mbar_fence_init();
    }
    if (tid < ER_LMAX) {
        const float l = (float)(tid > 0 ? tid : 1);
        coef[tid] = (2.f * l - 1.f) / l;
        coef[ER_LMAX + tid] = (l - 1.f) / l;
        coef[2 * ER_LMAX + tid] = (2.f * tid + 1.f) * 0.07957747154594767f;
    }
    if (a.geo_smem)
        for (int idx = tid; idx < a.geo_bytes / 4; idx += ER_NT) geo_s[idx] = a.p.geo[idx];
    __syncthreads();

    const bool graph_ok = (*a.status == 0);
    const long long nitems = a.nodes * nblk;
    int slot = 0;
    uint32_t phase = 0;

    if (warp == ER_CONS / 32) {
        // =============================== producer warp ===============================
        for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
            const long long i = item / nblk;
            const int kc0 = (int)(item - i * nblk) * cb;
            const int ncb = (Cpar - kc0 < cb) ? (Cpar - kc0) : cb;
            const int nsb = (ncb + cs - 1) / cs;
            const long long e_begin = graph_ok ? a.row_ptr[i] : 0, e_end = graph_ok ? a.row_ptr[i + 1] : 0;
            for (long long e0 = e_begin; e0 < e_end; e0 += 32) {
                const int n = (int)((e_end - e0 < 32) ? (e_end - e0) : 32);
                const long long s_mine = (lane < n) ? a.snd[e0 + lane] : 0;
                for (int el = 0; el < n; ++el) {
                    const long long s = __shfl_sync(0xffffffffu, s_mine, el);
                    if (lane == 0) {
                        const float* src = a.G + ((size_t)s * Cpar + kc0) * NF * UVp;
                        for (int sb = 0; sb < nsb; ++sb) {
                            const int ncs = (ncb - sb * cs < cs) ? (ncb - sb * cs) : cs;
                            const uint32_t bytes = (uint32_t)ncs * NF * UVp * 4u;
                            mbar_wait(&empty[slot], phase ^ 1u);
                            mbar_arrive_expect_tx(&full[slot], bytes);
                            tma_load_1d(ring + (size_t)slot * a.stage_bytes, src + (size_t)sb * cs * NF * UVp, bytes,
                                        &full[slot]);
                            if (++slot == NST) { slot = 0; phase ^= 1u; }
                        }
                    }
                }
            }
        }
        return;
    }

    // ================================= consumer warps =================================
    constexpr int QT = 1;
    int chl[NA], qd[QT];
    bool qok[QT];
    {
        const int cg = tid / QP;
        qd[0] = tid - cg * QP;
        qok[0] = cg < a.G_;
#pragma unroll
        for (int x = 0; x < NA; ++x) chl[x] = x * a.G_ + cg;
    }
    const float* geo = a.geo_smem ? geo_s : a.p.geo;
    const int lmax = a.p.lmax;

    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        const long long i = item / nblk;
        const int kc0 = (int)(item - i * nblk) * cb;
        const int ncb = (Cpar - kc0 < cb) ? (Cpar - kc0) : cb;
        const int nsb = (ncb + cs - 1) / cs;
        const long long e_begin = graph_ok ? a.row_ptr[i] : 0, e_end = graph_ok ? a.row_ptr[i + 1] : 0;

        float2 acc[NSBT][NA][2];
#pragma unroll
        for (int sb = 0; sb < NSBT; ++sb)
#pragma unroll
            for (int x = 0; x < NA; ++x) acc[sb][x][0] = acc[sb][x][1] = make_float2(0.f, 0.f);

        for (long long e0 = e_begin; e0 < e_end; e0 += a.EC) {
            const int ne = (int)((e_end - e0 < a.EC) ? (e_end - e0) : a.EC);
            // ---- M3: edge fields of the chunk on the grid (Eq.(48),(50); addition theorem, R12):
            // K(t) = sum_l (2l+1)/(4 pi) P_l(t), K'(t) likewise with P'_l = t P'_{l-1} + l P_{l-1}, t = r_e . Omega
            for (int idx = tid; idx < ne * UVp; idx += ER_CONS) {
                const int el = idx / UVp, q = idx - el * UVp;
                const long long e = e0 + el;
                float k0 = 0.f, k1 = 0.f;
                if (q < a.p.UV) {
                    float ex = a.edge_vec[3 * e], ey = a.edge_vec[3 * e + 1], ez = a.edge_vec[3 * e + 2];
                    const float rn = rsqrtf(ex * ex + ey * ey + ez * ez);
                    ex *= rn; ey *= rn; ez *= rn;
                    const float t = ex * geo[q] + ey * geo[UVp + q] + ez * geo[2 * UVp + q];
                    float pm = 1.f, pc = t, dc = 1.f;
                    float ks = coef[2 * ER_LMAX], kd = 0.f;
                    if (lmax >= 1) { ks = fmaf(coef[2 * ER_LMAX + 1], pc, ks); kd = coef[2 * ER_LMAX + 1]; }
                    for (int l = 2; l <= lmax; ++l) {
                        const float pn = fmaf(coef[l] * t, pc, -(coef[ER_LMAX + l] * pm));
                        const float c = coef[2 * ER_LMAX + l];
                        if (!ODD) {
                            ks = fmaf(c, pn, ks);
                        } else {
                            const float dn = fmaf(t, dc, (float)l * pc);
                            kd = fmaf(c, dn, kd);
                            dc = dn;
                        }
                        pm = pc; pc = pn;
                    }
                    if (!ODD) {
                        k0 = ks;
                    } else {
                        const float dth = ex * geo[3 * UVp + q] + ey * geo[4 * UVp + q] + ez * geo[5 * UVp + q];
                        const float dph = ex * geo[6 * UVp + q] + ey * geo[7 * UVp + q];
                        k0 = kd * dth;
                        k1 = -(kd * dph);  // stored negated: {E,I} = E_theta I_phi + (-E_phi) I_theta
                    }
                }
                Kbuf[((size_t)el * NF) * UVp + q] = k0;
                if (ODD) Kbuf[((size_t)el * NF + 1) * UVp + q] = k1;
            }
            for (int idx = tid; idx < ne * ncb; idx += ER_CONS) {
                const int el = idx / ncb, k = idx - el * ncb;
                Rbuf[el * cb + k] = a.edge_radial[(e0 + el) * a.C + a.perm_par[kc0 + k]];
            }
            consumer_sync();

            // ---- M4: staged sender grid x edge field, accumulated in fixed edge order
            for (int el = 0; el < ne; ++el) {
                const float4* k4 = reinterpret_cast<const float4*>(Kbuf + (size_t)el * NF * UVp);
                const float* rrow = Rbuf + el * cb;
                float4 kr[QT][NF];
#pragma unroll
                for (int j = 0; j < QT; ++j) {
                    kr[j][0] = k4[qd[j]];
                    if (ODD) kr[j][NF - 1] = k4[QP + qd[j]];
                }
#pragma unroll
                for (int sb = 0; sb < NSBT; ++sb) {
                    if (sb < nsb) {
                        const int ncs = (ncb - sb * cs < cs) ? (ncb - sb * cs) : cs;
                        const float4* g4 = reinterpret_cast<const float4*>(ring + (size_t)slot * a.stage_bytes);
                        mbar_wait(&full[slot], phase);
#pragma unroll
                        for (int x = 0; x < NA; ++x) {
                            constexpr int j = 0;
                            if (chl[x] < ncs && qok[j]) {
                                const float r = rrow[sb * cs + chl[x]];
                                if (!ODD) {
                                    const float4 g = g4[chl[x] * QP + qd[j]];
                                    const float2 p0 = __fmul2_rn(lo2(kr[j][0]), lo2(g));
                                    const float2 p1 = __fmul2_rn(hi2(kr[j][0]), hi2(g));
                                    acc[sb][x][0] = __ffma2_rn(p0, make_float2(r, r), acc[sb][x][0]);
                                    acc[sb][x][1] = __ffma2_rn(p1, make_float2(r, r), acc[sb][x][1]);
                                } else {
                                    // {E, I} = E_theta I_phi - E_phi I_theta   (edge = factor 1, Eq.(57))
                                    const float4 g0 = g4[chl[x] * 2 * QP + qd[j]], g1 = g4[chl[x] * 2 * QP + QP + qd[j]];
                                    float2 p0 = __fmul2_rn(lo2(kr[j][0]), lo2(g1));
                                    float2 p1 = __fmul2_rn(hi2(kr[j][0]), hi2(g1));
                                    p0 = __ffma2_rn(lo2(kr[j][NF - 1]), lo2(g0), p0);
                                    p1 = __ffma2_rn(hi2(kr[j][NF - 1]), hi2(g0), p1);
                                    acc[sb][x][0] = __ffma2_rn(p0, make_float2(r, r), acc[sb][x][0]);
                                    acc[sb][x][1] = __ffma2_rn(p1, make_float2(r, r), acc[sb][x][1]);
                                }
                            }
                        }
                        __syncwarp();
                        if (lane == 0) mbar_arrive(&empty[slot]);
                        if (++slot == NST) { slot = 0; phase ^= 1u; }
                    }
                }
            }
            consumer_sync();  // Kbuf / Rbuf are rewritten by the next chunk
        }

        // ---- pooled grid of this receiver (zeros for a receiver without in-edges)
#pragma unroll
        for (int sb = 0; sb < NSBT; ++sb) {
            if (sb < nsb) {
                const int ncs = (ncb - sb * cs < cs) ? (ncb - sb * cs) : cs;
                float4* sdst = reinterpret_cast<float4*>(a.S + ((size_t)i * Cpar + kc0 + sb * cs) * UVp);
#pragma unroll
                for (int x = 0; x < NA; ++x) {
                    constexpr int j = 0;
                    if (chl[x] < ncs && qok[j])
                        sdst[chl[x] * QP + qd[j]] =
                            make_float4(acc[sb][x][0].x, acc[sb][x][0].y, acc[sb][x][1].x, acc[sb][x][1].y);
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Host
// ------------------------------------------------------------------------------------------------
static int er_num_sms()
{
    static int n = 0;
    if (!n) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
        if (n <= 0) n = 148;
    }
    return n;
}

template <bool ODD, int NSBT, int NA>
static int launch_ring_t(const EdgeRingArgs& a, size_t smem, int grid, cudaStream_t st)
{
    auto kern = edge_ring_kernel<ODD, NSBT, NA>;
    CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<grid, ER_NT, smem, st>>>(a);
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

// *handled = false when the plan does not fit the ring kernel (the caller falls back to edge_kernel).
int launch_edge_ring(const Plan* p, bool odd, const float* G, const int64_t* row_ptr, const int64_t* edge_index,
                     int64_t E, const float* edge_vec, const float* edge_radial, const int* perm_par, int Cpar, int C,
                     float* S, int64_t nodes, const int32_t* status, cudaStream_t st, bool* handled)
{
    *handled = false;
    (void)E;
    if (Cpar <= 0 || nodes <= 0) return CGTP_OK;
    if (p->lmax >= ER_LMAX) return CGTP_OK;
    const int nf = odd ? 2 : 1;
    const int QP = p->UVp / 4;
    if (QP > ER_CONS) return CGTP_OK;  // cannot happen for band limits <= 20 (QP <= 473)
    const int G_ = ER_CONS / QP;
    // even kernel: 4 accumulators per thread and sub-block; 6 when that turns the whole channel set into one
    // sub-block (one ring stage per edge: configs[2] all-even 225 -> 192 us), measured slower otherwise
    int NA = odd ? 2 : 4;
    if (!odd && Cpar > 4 * G_ && Cpar <= 6 * G_ && (size_t)6 * G_ * p->UVp * 4 * 3 <= 150 * 1024) NA = 6;
    const int cs_max = NA * G_;
    const int NSB_MAX = 12 / NA;  // NA * NSBT <= 12 float4 accumulators per thread
    // channel blocks: as few as possible with at most NSB_MAX sub-blocks each
    const int cb_max = cs_max * NSB_MAX;
    const int nblk = (Cpar + cb_max - 1) / cb_max;
    const int cb = (Cpar + nblk - 1) / nblk;
    int nsb = (cb + cs_max - 1) / cs_max;
    int cs = (cb + nsb - 1) / nsb;  // balanced sub-blocks
    cs = std::min(cs_max, (cs + G_ - 1) / G_ * G_);  // whole channel groups
    nsb = (cb + cs - 1) / cs;
    int nsbt = nsb <= 1 ? 1 : nsb <= 2 ? 2 : nsb <= 3 ? 3 : nsb <= 4 ? 4 : 6;

    const size_t budget = 200 * 1024;
    const size_t stage_bytes = (size_t)cs * nf * p->UVp * 4;
    size_t geo_bytes = (size_t)(odd ? 8 : 3) * p->UVp * 4;
    const int geo_smem = geo_bytes <= 32 * 1024 ? 1 : 0;
    if (!geo_smem) geo_bytes = 0;
    int EC = 8;
    while (EC > 1 && (size_t)EC * nf * p->UVp * 4 > 40 * 1024) EC >>= 1;
    const size_t k_bytes = (size_t)EC * nf * p->UVp * 4;
    const size_t r_bytes = (size_t)round_up(EC * cb, 4) * 4;
    const size_t fixed = 256 + 3 * ER_LMAX * 4 + geo_bytes + k_bytes + r_bytes;
    if (fixed + 2 * stage_bytes > budget) return CGTP_OK;
    int NST = (int)((budget - fixed) / stage_bytes);
    if (NST > ER_MAXST) NST = ER_MAXST;
    if (stage_bytes >= (1u << 20)) return CGTP_OK;  // mbarrier tx-count field

    EdgeRingArgs a;
    a.p = *p;
    a.G = G;
    a.row_ptr = row_ptr;
    a.snd = edge_index;
    a.edge_vec = edge_vec;
    a.edge_radial = edge_radial;
    a.perm_par = perm_par;
    a.S = S;
    a.status = status;
    a.nodes = nodes;
    a.Cpar = Cpar;
    a.C = C;
    a.cb = cb;
    a.nblk = nblk;
    a.cs = cs;
    a.G_ = G_;
    a.EC = EC;
    a.NST = NST;
    a.geo_smem = geo_smem;
    a.stage_bytes = (int)stage_bytes;
    a.k_bytes = (int)k_bytes;
    a.r_bytes = (int)r_bytes;
    a.geo_bytes = (int)geo_bytes;
    const size_t smem = fixed + (size_t)NST * stage_bytes;
    const int64_t nitems = nodes * nblk;
    const int grid = (int)std::min<int64_t>(nitems, er_num_sms());

    LaunchScope scope(odd ? K_EDGE_ODD : K_EDGE_EVEN, st);
    int rc = CGTP_OK;
    if (odd) {
        switch (nsbt) {
        case 1: rc = launch_ring_t<true, 1, 2>(a, smem, grid, st); break;
        case 2: rc = launch_ring_t<true, 2, 2>(a, smem, grid, st); break;
        case 3: rc = launch_ring_t<true, 3, 2>(a, smem, grid, st); break;
        case 4: rc = launch_ring_t<true, 4, 2>(a, smem, grid, st); break;
        default: rc = launch_ring_t<true, 6, 2>(a, smem, grid, st); break;
        }
    } else {
        if (NA == 6) {
            rc = launch_ring_t<false, 1, 6>(a, smem, grid, st);
        } else {
            switch (nsbt) {
            case 1: rc = launch_ring_t<false, 1, 4>(a, smem, grid, st); break;
            case 2: rc = launch_ring_t<false, 2, 4>(a, smem, grid, st); break;
            default: rc = launch_ring_t<false, 3, 4>(a, smem, grid, st); break;
            }
        }
    }
    if (rc == CGTP_OK) *handled = true;
    return rc;
}

}  // namespace cgtp
