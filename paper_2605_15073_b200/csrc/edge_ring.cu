// edge_ring.cu -- rows M3 + M4 of SURVEY.md 8(a) (edge factor, gather, product / surface-curl pairing,
// neighbour sum; Eq.(48),(50),(52) :402-:415, Eq.(57) :443) as a persistent, warp-specialised
// streaming kernel:
//   * one CTA per SM loops over (receiver, channel block) items; a producer warp walks the receiver's
//     in-edges and streams the sender's grid block from HBM into a shared-memory ring with TMA bulk
//     copies (cp.async.bulk + mbarrier complete_tx), one stage = one (edge, channel sub-block) span,
//     contiguous and 16-byte aligned in the G layout of message.cu;
//   * sixteen consumer warps evaluate the channel-independent edge field(s) K_e on the grid (Legendre
//     recurrence in r_e . Omega, chunks of edges, two edges per packed operation), multiply them and R~[e,c]
//     with the staged sender VALUE grid and accumulate in registers in input edge order -- deterministic, no
//     floating-point atomics; odd channels pair the value grid with (d_theta K_e, -(1/sin) d_phi K_e) into two
//     pooled grids, the derivatives of Y_lm being applied by the analysis (curl pairing by parts);
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
constexpr int ER_HDR = 256 + ER_LMAX * 16 + 8 * 16;  // barriers, coefficient table, edge unit vectors

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
    float4* coef = reinterpret_cast<float4*>(smem + 256);  // [ER_LMAX]: (2l-1)/l, -(l-1)/l, (2l+1)/(4 pi), l
    float4* Ebuf = coef + ER_LMAX;                         // [8]: unit vectors of the chunk's edges
    float* geo_s = reinterpret_cast<float*>(Ebuf + 8);
    float* Kbuf = reinterpret_cast<float*>(smem + ER_HDR + a.geo_bytes);  // [EC][NF][UVp]
    float* Rbuf = Kbuf + a.k_bytes / 4;                                                   // [EC][cb]
    unsigned char* ring = reinterpret_cast<unsigned char*>(Rbuf) + a.r_bytes;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int UVp = a.p.UVp, QP = UVp / 4;
    const int NST = a.NST, cs = a.cs, cb = a.cb, nblk = a.nblk, Cpar = a.Cpar;

    pdl_launch_dependents();  // programmatic dependent launch, common.cuh: barriers, recurrence coefficients and the plan's
                              // grid geometry below are independent of every earlier kernel
    if (tid == 0) {
        for (int s = 0; s < NST; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], ER_CONS / 32);
        }
        mbar_fence_init();
    }
    if (tid < ER_LMAX) {
        const float l = (float)(tid > 0 ? tid : 1);
        coef[tid] = make_float4((2.f * l - 1.f) / l, -(l - 1.f) / l, (2.f * tid + 1.f) * 0.07957747154594767f, l);
    }
    if (a.geo_smem)
        for (int idx = tid; idx < a.geo_bytes / 4; idx += ER_NT) geo_s[idx] = a.p.geo[idx];
    __syncthreads();

    pdl_wait();  // status / row_ptr (M0), G (M2) and the caller's edge arrays; S may still be read by an earlier kernel
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
                        const float* src = a.G + ((size_t)s * Cpar + kc0) * UVp;
                        for (int sb = 0; sb < nsb; ++sb) {
                            const int ncs = (ncb - sb * cs < cs) ? (ncb - sb * cs) : cs;
                            const uint32_t bytes = (uint32_t)ncs * UVp * 4u;
                            mbar_wait(&empty[slot], phase ^ 1u);
                            mbar_arrive_expect_tx(&full[slot], bytes);
                            tma_load_1d(ring + (size_t)slot * a.stage_bytes, src + (size_t)sb * cs * UVp, bytes,
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

        float2 acc[NSBT][NA][NF][2];
#pragma unroll
        for (int sb = 0; sb < NSBT; ++sb)
#pragma unroll
            for (int x = 0; x < NA; ++x)
#pragma unroll
                for (int f = 0; f < NF; ++f) acc[sb][x][f][0] = acc[sb][x][f][1] = make_float2(0.f, 0.f);

        // unit vectors of a chunk's edges (only the direction of edge_vec is used, R11)
        auto load_edges = [&](long long e0, long long e_end_) {
            const int n = (int)((e_end_ - e0 < a.EC) ? (e_end_ - e0) : a.EC);
            if (tid < n) {
                const long long e = e0 + tid;
                const float ex = a.edge_vec[3 * e], ey = a.edge_vec[3 * e + 1], ez = a.edge_vec[3 * e + 2];
                const float rn = rsqrtf(ex * ex + ey * ey + ez * ez);
                Ebuf[tid] = make_float4(ex * rn, ey * rn, ez * rn, 0.f);
            }
        };
        if (e_begin < e_end) {
            load_edges(e_begin, e_end);
            consumer_sync();
        }

        for (long long e0 = e_begin; e0 < e_end; e0 += a.EC) {
            const int ne = (int)((e_end - e0 < a.EC) ? (e_end - e0) : a.EC);
            // ---- M3: edge fields of the chunk on the grid (Eq.(48),(50); addition theorem, R12):
            // K(t) = sum_l (2l+1)/(4 pi) P_l(t), K'(t) likewise with P'_l = t P'_{l-1} + l P_{l-1}, t = r_e . Omega.
            // Two edges per work item in the halves of packed FP32 operations.
            {
                // work items = (edge pair, grid point), dealt over all consumer threads
                const int total = ((ne + 1) >> 1) * UVp;
                {
                    {
                        for (int w = tid; w < total; w += ER_CONS) {
                            const int pr = w / UVp, q = w - pr * UVp;
                            const int el = 2 * pr;
                            const bool live = q < a.p.UV;
                            const float gx = geo[q], gy = geo[UVp + q], gz = geo[2 * UVp + q];
                            float tx = 0.f, ty = 0.f, tz = 0.f, fx = 0.f, fy = 0.f;
                            if (ODD) {
                                tx = geo[3 * UVp + q]; ty = geo[4 * UVp + q]; tz = geo[5 * UVp + q];
                                fx = geo[6 * UVp + q]; fy = geo[7 * UVp + q];
                            }
                            const int el1 = (el + 1 < ne) ? el + 1 : el;
                            const float4 ea = Ebuf[el], eb = Ebuf[el1];
                            const float2 t = make_float2(fmaf(ea.x, gx, fmaf(ea.y, gy, ea.z * gz)),
                                                         fmaf(eb.x, gx, fmaf(eb.y, gy, eb.z * gz)));
                            float2 pm = make_float2(1.f, 1.f), pc = t, dc = make_float2(1.f, 1.f);
                            const float c0 = coef[0].z, c1 = coef[1].z;
                            float2 ks = make_float2(c0, c0), kd = make_float2(0.f, 0.f);
                            if (lmax >= 1) {
                                ks = __ffma2_rn(make_float2(c1, c1), pc, ks);
                                kd = make_float2(c1, c1);
                            }
                            for (int l = 2; l <= lmax; ++l) {
                                const float4 c = coef[l];
                                const float2 pn = __ffma2_rn(make_float2(c.x, c.x), __fmul2_rn(t, pc),
                                                             __fmul2_rn(make_float2(c.y, c.y), pm));
                                if (!ODD) {
                                    ks = __ffma2_rn(make_float2(c.z, c.z), pn, ks);
                                } else {
                                    const float2 dn = __ffma2_rn(t, dc, __fmul2_rn(make_float2(c.w, c.w), pc));
                                    kd = __ffma2_rn(make_float2(c.z, c.z), dn, kd);
                                    dc = dn;
                                }
                                pm = pc; pc = pn;
                            }
                            float2 k0 = ks, k1 = make_float2(0.f, 0.f);
                            if (ODD) {
                                const float2 dth = make_float2(fmaf(ea.x, tx, fmaf(ea.y, ty, ea.z * tz)),
                                                               fmaf(eb.x, tx, fmaf(eb.y, ty, eb.z * tz)));
                                const float2 dph = make_float2(fmaf(ea.x, fx, ea.y * fy), fmaf(eb.x, fx, eb.y * fy));
                                k0 = __fmul2_rn(kd, dth);
                                k1 = __fmul2_rn(kd, make_float2(-dph.x, -dph.y));  // stored negated (X1 = -sum R~ E_phi I)
                            }
                            if (!live) k0 = k1 = make_float2(0.f, 0.f);
                            Kbuf[((size_t)el * NF) * UVp + q] = k0.x;
                            if (ODD) Kbuf[((size_t)el * NF + 1) * UVp + q] = k1.x;
                            if (el1 != el) {
                                Kbuf[((size_t)el1 * NF) * UVp + q] = k0.y;
                                if (ODD) Kbuf[((size_t)el1 * NF + 1) * UVp + q] = k1.y;
                            }
                        }
                    }
                }
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
                                const float4 g = g4[chl[x] * QP + qd[j]];
                                if (!ODD) {
                                    const float2 p0 = __fmul2_rn(lo2(kr[j][0]), lo2(g));
                                    const float2 p1 = __fmul2_rn(hi2(kr[j][0]), hi2(g));
                                    acc[sb][x][0][0] = __ffma2_rn(p0, make_float2(r, r), acc[sb][x][0][0]);
                                    acc[sb][x][0][1] = __ffma2_rn(p1, make_float2(r, r), acc[sb][x][0][1]);
                                } else {
                                    // surface-curl pairing by parts: the sender's VALUE field is
                                    // gathered once and paired with both derivative fields of the edge,
                                    // X0 += R~ E_theta I,  X1 += R~ (-E_phi) I; the analysis applies {., Y_lm}
                                    const float2 g0 = __fmul2_rn(lo2(g), make_float2(r, r));
                                    const float2 g1 = __fmul2_rn(hi2(g), make_float2(r, r));
                                    acc[sb][x][0][0] = __ffma2_rn(lo2(kr[j][0]), g0, acc[sb][x][0][0]);
                                    acc[sb][x][0][1] = __ffma2_rn(hi2(kr[j][0]), g1, acc[sb][x][0][1]);
                                    acc[sb][x][NF - 1][0] = __ffma2_rn(lo2(kr[j][NF - 1]), g0, acc[sb][x][NF - 1][0]);
                                    acc[sb][x][NF - 1][1] = __ffma2_rn(hi2(kr[j][NF - 1]), g1, acc[sb][x][NF - 1][1]);
                                }
                            }
                        }
                        __syncwarp();
                        if (lane == 0) mbar_arrive(&empty[slot]);
                        if (++slot == NST) { slot = 0; phase ^= 1u; }
                    }
                }
            }
            if (e0 + a.EC < e_end) load_edges(e0 + a.EC, e_end);  // Ebuf was last read before the first sync of this chunk
            consumer_sync();  // Kbuf / Rbuf are rewritten by the next chunk
        }

        // ---- pooled grid of this receiver (zeros for a receiver without in-edges)
#pragma unroll
        for (int sb = 0; sb < NSBT; ++sb) {
            if (sb < nsb) {
                const int ncs = (ncb - sb * cs < cs) ? (ncb - sb * cs) : cs;
                float4* sdst = reinterpret_cast<float4*>(a.S + ((size_t)i * Cpar + kc0 + sb * cs) * NF * UVp);
#pragma unroll
                for (int x = 0; x < NA; ++x) {
                    constexpr int j = 0;
                    if (chl[x] < ncs && qok[j]) {
#pragma unroll
                        for (int f = 0; f < NF; ++f)
                            sdst[(chl[x] * NF + f) * QP + qd[j]] = make_float4(acc[sb][x][f][0].x, acc[sb][x][f][0].y,
                                                                               acc[sb][x][f][1].x, acc[sb][x][f][1].y);
                    }
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Host
// ------------------------------------------------------------------------------------------------

template <bool ODD, int NSBT, int NA>
static int launch_ring_t(const EdgeRingArgs& a, size_t smem, int grid, cudaStream_t st)
{
    auto kern = edge_ring_kernel<ODD, NSBT, NA>;
    CGTP_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CGTP_CUDA_CHECK(launch_pdl(kern, (unsigned)grid, (unsigned)ER_NT, smem, st, a));
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
    // odd: two accumulator fields per channel (X0, X1), so NA * NSBT <= 6: channel blocks of up to 6 G_ channels, as
    // one sub-block of 6 per thread when a block needs more than 3 G_ (configs[4]: 10.0 -> 9.4 ms), else 3 per thread
    int NA = odd ? 3 : 4;
    if (odd) {
        const int nb = (Cpar + 6 * G_ - 1) / (6 * G_);
        if ((Cpar + nb - 1) / nb > 3 * G_) NA = 6;
    }
    if (!odd && Cpar > 4 * G_ && Cpar <= 6 * G_ && (size_t)6 * G_ * p->UVp * 4 * 3 <= 150 * 1024) NA = 6;
    const int cs_max = NA * G_;
    const int NSB_MAX = (odd ? 6 : 12) / NA;  // at most 12 float4 accumulators per thread
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
    const size_t stage_bytes = (size_t)cs * p->UVp * 4;  // one gathered field per channel for both parities
    size_t geo_bytes = (size_t)(odd ? 8 : 3) * p->UVp * 4;
    const int geo_smem = geo_bytes <= 32 * 1024 ? 1 : 0;
    if (!geo_smem) geo_bytes = 0;
    int EC = 8;
    while (EC > 1 && (size_t)EC * nf * p->UVp * 4 > 40 * 1024) EC >>= 1;
    const size_t k_bytes = (size_t)EC * nf * p->UVp * 4;
    const size_t r_bytes = (size_t)round_up(EC * cb, 4) * 4;
    const size_t fixed = ER_HDR + geo_bytes + k_bytes + r_bytes;
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
    const int grid = (int)std::min<int64_t>(nitems, num_sms());

    LaunchScope scope(odd ? K_EDGE_ODD : K_EDGE_EVEN, st);
    int rc = CGTP_OK;
    if (odd) {
        if (NA == 3) {
            rc = nsbt <= 1 ? launch_ring_t<true, 1, 3>(a, smem, grid, st) : launch_ring_t<true, 2, 3>(a, smem, grid, st);
        } else if (NA == 6) {
            rc = launch_ring_t<true, 1, 6>(a, smem, grid, st);
        } else {
            rc = nsbt <= 1 ? launch_ring_t<true, 1, 2>(a, smem, grid, st)
               : nsbt <= 2 ? launch_ring_t<true, 2, 2>(a, smem, grid, st)
                           : launch_ring_t<true, 3, 2>(a, smem, grid, st);
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
