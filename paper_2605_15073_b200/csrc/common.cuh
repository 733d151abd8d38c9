// common.cuh -- shared host/device declarations of libcgtp (sm_100a only).
#pragma once

#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <vector>

#include "../../include/cgtp.h"

namespace cgtp {

// Band limits with a compiled kernel instantiation; max(lmax, lmax_out) is rounded up to the next one
// (the extra coefficient rows are zero).  CGTP_FOR_EACH_BAND(X) expands X(LB) for each of them.
#define CGTP_FOR_EACH_BAND(X) X(1) X(2) X(3) X(4) X(5) X(6) X(8) X(10) X(12) X(16) X(20)
constexpr int kMaxBand = 20;
inline int kernel_band(int b)
{
    const int bands[] = {1, 2, 3, 4, 5, 6, 8, 10, 12, 16, 20};
    for (int v : bands)
        if (b <= v) return v;
    return -1;
}

// Ordinal of the calling thread's current CUDA device (-1 on error).  The plan / table / scratch caches hold device
// pointers, so each of them is keyed by this ordinal: a process that drives several GPUs gets one entry per device.
inline int current_device()
{
    int d = -1;
    return cudaGetDevice(&d) == cudaSuccess ? d : -1;
}
// Multiprocessor count of the current device (cached per ordinal).
int num_sms();

// Test-only kernel-path switch (cgtp_set_kernel_path): bit set = take the generic kernel where a specialised one exists.
enum : int { PATH_GENERIC_CORE = 1, PATH_GENERIC_EDGE = 2, PATH_GENERIC_PROJ = 4, PATH_GENERIC_SYNTH = 8, PATH_UNFUSED_ONSITE = 16, PATH_FUSED_ONSITE = 32, PATH_FIELD_PER_EDGE = 64, PATH_SMEM_CORE = 128, PATH_PLAIN_LAUNCH = 256 };
int kernel_path();
void set_kernel_path(int flags);

__host__ __device__ constexpr int round_up(int x, int m) { return (x + m - 1) / m * m; }
__host__ __device__ constexpr int tri_index(int l, int m) { return l * (l + 1) / 2 + m; }

// ---------------------------------------------------------------------------------------------
// Plan: quadrature grid + FP32 device tables for one (lmax, lmax_out).  Built once in FP64 on the
// host (tables.cu), cached for the life of the process.
//
// Grid (R8): U Gauss-Legendre nodes x_u = cos(theta_u) (u = 0 is the
// northernmost, x_{U-1-u} = -x_u), V azimuths phi_v = 2 pi v / V.
// Folding: only the northern half u' < Uh = ceil(U/2) of the Legendre tables and only
// v' < Vh = V/2 + 1 of the Fourier tables are stored; the southern / mirrored halves follow from
// P~_l^m(-x) = (-1)^(l+m) P~_l^m(x) and cos/sin(m (2pi - phi)).
// ---------------------------------------------------------------------------------------------
struct Plan {
    int dev;   // CUDA device ordinal the tables live on: every cache of the library is keyed by it
    int lmax, lmax_out;
    int nu;    // body order the grid is exact for (2 everywhere except the nu-body entry point)
    int LB;    // kernel band limit = kernel_band(max(lmax, lmax_out)); tables cover 0 <= m <= l <= LB
    int U, V;  // grid
    int Uh, Vh;
    int UV, UVp;  // U*V and U*V rounded up to a multiple of 4 floats (16 bytes)
    int NTRI;     // (LB+1)(LB+2)/2 rounded up to a multiple of 4: row length of the Legendre tables
    int QSTR;     // LB+1 rounded up to a multiple of 4: row length of the Fourier tables
    int L2, L2p, Lo2, Lo2p;  // (lmax+1)^2, (lmax_out+1)^2 and their multiples of 4
    // Legendre tables, [Uh][NTRI], entry tri_index(l,m):
    const float* PT;  // P~_l^m(x_u)                          (p_ulm of Eq.(22))
    const float* DT;  // d/dtheta P~_l^m(cos theta) at theta_u (theta-form of d_x p_ulm, :445)
    const float* ST;  // m P~_l^m(x_u) / sin(theta_u)         ((1/sin theta) d_phi of Eq.(11), :107)
    const float* WP;  // w_u P~_l^m(x_u), equator row halved  (Eq.(40), :342)
    const float* WD;  // w_u d/dtheta P~_l^m, equator row halved      (analysis of the by-parts curl pairing, M5 odd)
    const float* WS;  // w_u m P~_l^m / sin(theta), equator row halved
    // Fourier tables (real form, Eq.(C2) :668), [Vh][QSTR]:
    const float* QC;  // QC[v'][0] = 1, QC[v'][m] = sqrt2 cos(m phi_v')
    const float* QS;  // QS[v'][m] = sqrt2 sin(m phi_v'), zero for m = 0 and for self-mirrored v'
    const float* WV;  // [round_up(Vh,4)]: (2 pi / V), halved for self-mirrored v'   (Eq.(39), :339)
    // Grid geometry for the edge factor, [8][UVp]: Omega_xyz, theta_hat_xyz, phi_hat_xy (zero padded)
    const float* geo;
    // host copies of QC, QS, WV: kernels that take the azimuthal tables as kernel parameters (constant bank, read on the
    // uniform datapath instead of through shared memory) copy them from here
    const float *hQC, *hQS, *hWV;
};

// FP64 host helpers of the table builder (tables.cu), shared with the packed tables of onsite_core.cu.
void gauss_legendre(int U, std::vector<double>& x, std::vector<double>& w);
void legendre_values(int U, int LB, const std::vector<double>& x, std::vector<double>& P);  // P[u][l][m]

// Returns the cached plan, creating it on first use (cudaMalloc + blocking copies, once).
// nullptr + cgtp_last_error on failure.
const Plan* get_plan(int lmax, int lmax_out);
// Same with the grid of a nu-body product: U = ceil((nu lmax + lmax_out + 1)/2), V = nu lmax + lmax_out + 1
// ("Higher-body-order products tighten this requirement linearly in the body order nu").
const Plan* get_plan_nu(int lmax, int lmax_out, int nu);

// ---------------------------------------------------------------------------------------------
// Channel plan: parity_mask -> permutation that lists the even channels first (stable).
// ---------------------------------------------------------------------------------------------
struct ChannelPlan {
    int dev;
    int C, Ce, Co;
    const int* perm_dev;  // device [C]: perm[k] = original channel index of sorted position k
    int perm_host[1024];
};
const ChannelPlan* get_channel_plan(int C, const uint8_t* parity_mask);

// ---------------------------------------------------------------------------------------------
// Parity plan (parity.cu): weight-row / weight-column index tables of the passes of the parity-slot entry points.
// ---------------------------------------------------------------------------------------------
struct ParityPlan {
    int ordinal;     // CUDA device ordinal of `dev`
    int C, N;
    bool message;
    int npass;       // 4 on-site passes (s1, s2), 2 message passes (s_in)
    const int* dev;  // device [npass][2][4C]: idx_in, idx_out of pass ps
    const int* idx_in(int ps) const { return dev + (size_t)ps * 8 * C; }
    const int* idx_out(int ps) const { return dev + (size_t)ps * 8 * C + 4 * C; }
};
const ParityPlan* get_parity_plan(int C, int N, bool message);
// Clears T[col][lm] for the degrees l whose parity is not the sigma of the column's channel (Eq.(54)).
int launch_sigma_mask(float* T, int stride, int64_t ncols, int Cpar, int Cs, int Lo2, cudaStream_t st);

// ---------------------------------------------------------------------------------------------
// Errors, launch accounting, profiling
// ---------------------------------------------------------------------------------------------
void set_error(const char* fmt, ...);
void clear_error();

enum Kind {
    K_PROJ_IN = 0,
    K_ONSITE_EVEN,
    K_ONSITE_ODD,
    K_PROJ_OUT,
    K_SEGMENTS,
    K_NODE_SYNTH_EVEN,
    K_NODE_SYNTH_ODD,
    K_EDGE_EVEN,
    K_EDGE_ODD,
    K_ANALYSIS_EVEN,
    K_ANALYSIS_ODD,
    K_MISC,
    K_ONSITE_FUSED,
    K_COUNT
};

// RAII around one kernel launch: counts it and, when profiling is on, brackets it with events.
struct LaunchScope {
    LaunchScope(Kind kind, cudaStream_t stream);
    ~LaunchScope();
    Kind kind;
    cudaStream_t stream;
    void* rec;
};

#define CGTP_CUDA_CHECK(expr)                                                                    \
    do {                                                                                         \
        cudaError_t _e = (expr);                                                                 \
        if (_e != cudaSuccess) {                                                                 \
            ::cgtp::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__, __LINE__); \
            return CGTP_ERR_CUDA;                                                                \
        }                                                                                        \
    } while (0)

// ---------------------------------------------------------------------------------------------
// Programmatic dependent launch (the kernels of the four-launch on-site step and of message passing M1-M6): a kernel
// launched with launch_pdl may be
// scheduled while its predecessor in the stream is still running, once every CTA of the predecessor has executed
// pdl_launch_dependents() (or exited).  It may then run the part of its prologue that touches nothing the predecessor
// writes (tables, weights -> shared memory) and MUST execute pdl_wait() before its first access to such data: the wait
// returns when the predecessor grid has completed and its writes are visible.  Launched without the attribute both
// instructions are no-ops.  A successor is scheduled only after EVERY CTA of its predecessor has started (and signalled), so
// a waiting successor cannot keep a predecessor's CTA off an SM, whether or not the predecessor's grid is resident at once.
// ---------------------------------------------------------------------------------------------
// Per calling thread: true = launch_pdl launches in plain stream order.  Set for the duration of a call by the entry points
// whose steps are long (PdlScope): chaining pays where the kernel boundaries are a visible share of the step (configs[1]
// 0.240 -> 0.224 ms, configs[2] 0.521 -> 0.495 ms) and does not where the kernels run for milliseconds (configs[4]: 21.3 ms
// chained against 21.0 ms plain, medians of six alternating runs on a power-capped box).
bool pdl_plain();
void set_pdl_plain(bool plain);
struct PdlScope {
    explicit PdlScope(bool plain) : prev(pdl_plain()) { set_pdl_plain(plain); }
    ~PdlScope() { set_pdl_plain(prev); }
    bool prev;
};
// intermediate data of a step (bytes) above which its kernels are launched in plain order
constexpr size_t kPdlMaxBytes = (size_t)256 << 20;

#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), unsigned grid, unsigned block, size_t smem, cudaStream_t st, Args&&... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = ((kernel_path() & PATH_PLAIN_LAUNCH) || pdl_plain()) ? 0 : 1;  // test switch / long steps: plain order
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}
#endif

// ---------------------------------------------------------------------------------------------
// Stage launchers (one per row of SURVEY.md 8(a)); all asynchronous on `st`.
// ---------------------------------------------------------------------------------------------

// S1/S5/M1/M6: Out[b][m][j] = sum_{kk<K} W[widx_m(m)*ldw_m + widx_k(kk)*ldw_k] * X[b*x_bs + kk*x_rs + j]
// for j < J.  Rows m < m_split go to out0 + b*o_bs0 + m*o_rs, rows m >= m_split to
// out1 + b*o_bs1 + (m-m_split)*o_rs.  idx arrays may be nullptr (identity).
struct ProjArgs {
    const float* X;
    int64_t x_bs;
    int x_rs;
    const float* W;
    int ldw_m, ldw_k;
    const int* idx_m;
    const int* idx_k;
    int M, K, J;
    float* out0;
    int64_t o_bs0;
    float* out1;
    int64_t o_bs1;
    int m_split;
    int o_rs;
    int64_t batch;
    int accumulate;  // 1: add to the output instead of overwriting it (second pass of the parity-slot entry points)
    int j0;          // first column of every X row that is used: X[.. + j0 + j], j < J (l-dependent weights: one degree l
                     // per launch, j0 = l^2, J = 2l+1); the output pointers are given already offset by the caller
};
int launch_proj(const ProjArgs* args, int nargs, Kind kind, cudaStream_t st);
// Fast path of launch_proj (proj_fast.cu): TMA-staged features, packed FP32 FMAs; *handled = false when the
// layout conditions (even K, 16-byte aligned atom blocks, ...) do not hold and the generic kernel must run.
int launch_proj_fast(const ProjArgs* args, int nargs, Kind kind, cudaStream_t st, bool* handled);

// All degrees of an l-dependent-weight projection in one launch (proj_multi.cu); FP32 path only; *handled = false ->
// launch the problems one by one.
int launch_proj_multi(const ProjArgs* args, int nargs, Kind kind, cudaStream_t st, bool* handled);

// Tensor-core path of launch_proj (proj_tc.cu: tcgen05.mma kind::tf32, TMEM accumulators), taken only when
// the math mode is CGTP_MATH_3XTF32 / CGTP_MATH_TF32; *handled = false otherwise.
int launch_proj_tc(const ProjArgs* args, int nargs, Kind kind, cudaStream_t st, bool* handled);
void set_math_mode(int mode);
int get_math_mode();

// S2-S4 fused: T[col][lm] from Ha[col], Hb[col]; ncols columns of one parity.
// Generic kernel (any compiled band limit): H rows of stride p->L2p, T rows of stride p->Lo2p.
int launch_onsite_generic(const Plan* p, bool odd, const float* Ha, const float* Hb, float* T, int64_t ncols,
                          cudaStream_t st);
// Fast kernel (onsite_core.cu): lane = column, packed FP32 FMAs.  H rows of stride onsite_fast_hstride(p),
// T rows of stride onsite_fast_tstride(p) (both odd, so that lane-strided shared-memory accesses are
// conflict-free); the column count is padded up to a multiple of 32 in both buffers.
bool onsite_fast_supported(const Plan* p, bool odd);
inline int onsite_fast_hstride(const Plan* p) { return p->L2 | 1; }
inline int onsite_fast_tstride(const Plan* p) { return p->Lo2 | 1; }
int launch_onsite_fast(const Plan* p, bool odd, const float* Ha, const float* Hb, float* T, int64_t ncols,
                       cudaStream_t st);
// Register-resident core for small band limits (onsite_reg.cu): one thread per column, nothing exchanged between
// threads; same buffers and strides as the fast kernel, which hands the band limits of onsite_reg_supported() over to it
// unless CGTP_PATH_SMEM_CORE is set.  send / cpar / status as in launch_onsite_fast_field (cpar a multiple of 32).
bool onsite_reg_supported(const Plan* p, bool odd);
int launch_onsite_reg(const Plan* p, bool odd, const float* Ha, const float* Hb, float* T, int64_t ncols, cudaStream_t st,
                      const int64_t* send, int cpar, const int32_t* status);

// S1-S5 in one kernel (onsite_fused.cu): reads A, B once, writes out once, H and T stay in shared memory.  idx_in[k] = row
// of W_a / W_b of internal (parity-sorted) channel k; idx_out_e / idx_out_o = column of W_out of the even / odd channels;
// `out` must be the dense [batch][2][N][Lo2] block.  *handled = false when the shape does not fit (band limit > 8,
// lmax_out > lmax, shared memory): the caller runs the four-launch path.
int launch_onsite_fused(const Plan* p, int N, int C, int Ce, int Co, const float* A, const float* B, const float* W_a,
                        const float* W_b, const int* idx_in, const float* W_out, int ldw_out, const int* idx_out_e,
                        const int* idx_out_o, float* out, int64_t batch, cudaStream_t st, bool* handled);

// Same core with factor 2 read through the edge list (two-field coupling, Eq.(28)): column e * cpar + k of
// Ha pairs with column send[e] * cpar + k of Hn.  *handled = false when the kernel's group width does not divide cpar.
int launch_onsite_fast_gather(const Plan* p, bool odd, const float* Ha, const float* Hn, const int64_t* send, int cpar,
                              const int32_t* status, float* T, int64_t ncols, cudaStream_t st, bool* handled);

// Two-field coupling with the neighbour sum on the grid (onsite_core.cu, field_pool_core_kernel): see there.
int launch_field_pool_core(const Plan* p, bool odd, const float* Ha, const float* Hn, const int64_t* send,
                           const int64_t* row_ptr, int cpar, const int32_t* status, float* Tn, int64_t nodes, int64_t e0,
                           int64_t e1, cudaStream_t st, bool* handled);

// nu-body form of S2-S4 (nbody.cu): T[col][Lo2p] = analysis of prod_s synthesis(H[s][col]); H holds nu blocks at
// distance nbody_hfstride(p, ncols) floats, each [ncols][nbody_hstride(p)] (odd row stride), plus 4 rows of padding at
// the end; p a plan of get_plan_nu.  CGTP_ERR_UNSUPPORTED above band limit 8 or body order 4.
bool nbody_supported(int LB, int nu);
int nbody_hstride(const Plan* p);
int64_t nbody_hfstride(const Plan* p, int64_t ncols);
int launch_nbody(const Plan* p, const float* H, float* T, int64_t ncols, cudaStream_t st);
// Register-resident form for small band limits (nbody_reg.cu): one thread per column.  H: [nu][hfs] with rows of stride
// L2 | 1 and every factor block padded to whole groups of 32 columns; T rows of stride Lo2 | 1, padded likewise.
bool nbody_reg_supported(const Plan* p);
int launch_nbody_reg(const Plan* p, const float* H, int64_t hfs, float* T, int64_t ncols, cudaStream_t st);

// M0: row_ptr over `nodes` receivers; senders are validated against n_send
int launch_segments(const int64_t* edge_index, int64_t E, int64_t nodes, int64_t n_send, int64_t* row_ptr,
                    int32_t* status, cudaStream_t st);
// M2: value grid field of the projected node features, G[col][UVp], for the channels of either parity (`odd` only
// labels the launch for the profiler: the odd channels pair the edge's derivative fields with the sender's VALUE
// field and move the derivatives onto Y_lm in the analysis).
int launch_node_synth(const Plan* p, bool odd, const float* H, float* G, int64_t ncols, cudaStream_t st);
// Lane = column form of M2 (sht_fast.cu) for band limits whose 32-column tile fits shared memory: H rows of stride
// synth_fast_hstride(p) (odd), the H buffer padded to whole groups of 32 columns.
bool synth_fast_supported(const Plan* p);
inline int synth_fast_hstride(const Plan* p) { return p->L2 | 1; }
int launch_node_synth_fast(const Plan* p, bool odd, const float* H, int hstride, float* G, int64_t ncols, cudaStream_t st);
// M3+M4: channels of one parity.  even: S[i][kc][UVp] = sum_e R~ K_e G[send(e)];
// odd: S[i][kc][2][UVp] = sum_e R~ (d_theta K_e, -(1/sin) d_phi K_e) G[send(e)].
int launch_edge(const Plan* p, bool odd, const float* G, const int64_t* row_ptr, const int64_t* edge_index,
                int64_t E, const float* edge_vec, const float* edge_radial, const int* perm_par, int Cpar, int C,
                float* S, int64_t nodes, const int32_t* status, cudaStream_t st);
// Persistent TMA-ring form of launch_edge (edge_ring.cu); *handled = false -> use launch_edge's generic kernel.
int launch_edge_ring(const Plan* p, bool odd, const float* G, const int64_t* row_ptr, const int64_t* edge_index,
                     int64_t E, const float* edge_vec, const float* edge_radial, const int* perm_par, int Cpar, int C,
                     float* S, int64_t nodes, const int32_t* status, cudaStream_t st, bool* handled);
// M3+M4 with the l1-dependent radial factor edge_radial [E][C][lmax+1] (edge_lr.cu; Eq.(46)).
int launch_edge_lr(const Plan* p, bool odd, const float* G, const int64_t* row_ptr, const int64_t* edge_index, int64_t E,
                   const float* edge_vec, const float* edge_radial, const int* perm_par, int Cpar, int C, float* S,
                   int64_t nodes, const int32_t* status, cudaStream_t st);
// Two-field coupling (edge_field.cu; Eq.(28)): block gather Hb[e] = Hn[send[e]] and the pooled sum
// Tn[i] (+)= sum of T[e - e0] over the edges of receiver i inside [e0, e1); blocks of `blk` contiguous floats.
int launch_field_gather(const float* Hn, const int64_t* send, float* Hb, int64_t ne, int blk, const int32_t* status,
                        cudaStream_t st);
int launch_field_pool(const float* T, const int64_t* row_ptr, float* Tn, int64_t nodes, int64_t e0, int64_t e1, int blk,
                      const int32_t* status, cudaStream_t st);
// M5: T[col][Lo2p] = analysis of S[col][UVp] (even) or of the field pair S[col][2][UVp] against {., Y_lm} (odd)
int launch_analysis(const Plan* p, bool odd, const float* S, float* T, int64_t ncols, cudaStream_t st);

}  // namespace cgtp
