// api.cu -- the C ABI of include/cgtp.h: argument validation, workspace carving, stage sequencing.
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

#include "common.cuh"

namespace cgtp {
const char* last_error();
int64_t launch_count();
void profile_enable(bool on);
int profile_collect(double* ms, int64_t* launches);

static const char* kKindNames[K_COUNT] = {
    "proj_in",        "onsite_core_even", "onsite_core_odd", "proj_out",      "segments",      "node_synth_even",
    "node_synth_odd", "edge_even",        "edge_odd",        "analysis_even", "analysis_odd",  "misc",
    "onsite_fused"};

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
static inline int64_t round_up64(int64_t x, int64_t m) { return (x + m - 1) / m * m; }
static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

struct Carver {
    char* base;
    size_t off;
    explicit Carver(void* b) : base(static_cast<char*>(b)), off(0) {}
    template <class T>
    T* take(size_t count)
    {
        T* p = reinterpret_cast<T*>(base + off);
        off = align_up(off + count * sizeof(T), 256);
        return p;
    }
};

static int check_common(int lmax, int lmax_out, int N, int C, const uint8_t* mask)
{
    if (lmax < 0 || lmax_out < 0 || lmax_out > 2 * lmax) {
        set_error("invalid band limits lmax=%d lmax_out=%d (need 0 <= lmax_out <= 2*lmax)", lmax, lmax_out);
        return CGTP_ERR_INVALID;
    }
    if (N <= 0 || C <= 0) { set_error("N and C must be positive (N=%d, C=%d)", N, C); return CGTP_ERR_INVALID; }
    if (C > 1024) { set_error("C=%d exceeds the compiled limit 1024", C); return CGTP_ERR_UNSUPPORTED; }
    if (kernel_band(lmax > lmax_out ? lmax : lmax_out) < 0) {
        set_error("band limit max(lmax,lmax_out)=%d exceeds cgtp_max_lmax()=%d", lmax > lmax_out ? lmax : lmax_out, kMaxBand);
        return CGTP_ERR_UNSUPPORTED;
    }
    if (!mask) { set_error("parity_mask is NULL"); return CGTP_ERR_INVALID; }
    for (int c = 0; c < C; ++c)
        if (mask[c] > 1) { set_error("parity_mask[%d]=%d is not 0 or 1", c, (int)mask[c]); return CGTP_ERR_INVALID; }
    return CGTP_OK;
}

static size_t onsite_ws_bytes(int lmax, int lmax_out, int C, int64_t batch)
{
    const size_t L2p = round_up((lmax + 1) * (lmax + 1), 4), Lo2p = round_up((lmax_out + 1) * (lmax_out + 1), 4);
    // rows may use the odd strides of the fast core (<= L2p + 1) and columns are padded to groups of 32
    return ((size_t)batch * C + 64) * (2 * (L2p + 4) + (Lo2p + 4)) * sizeof(float) + 8 * 256;
}

static size_t message_ws_bytes(int lmax, int lmax_out, int C, int Co, int64_t n_send, int64_t n_recv)
{
    const size_t L2p = round_up((lmax + 1) * (lmax + 1), 4), Lo2p = round_up((lmax_out + 1) * (lmax_out + 1), 4);
    const int U = (2 * lmax + lmax_out + 2) / 2, V = 2 * lmax + lmax_out + 1;
    const size_t UVp = round_up(U * V, 4);
    // H, G (value grid, both parities) for the senders; S (two pooled grids per odd channel), T, row_ptr for the receivers
    // (H rows may use the odd stride of the fast synthesis, <= L2p + 1, with the columns padded to groups of 32)
    size_t fl = ((size_t)n_send * C + 64) * (L2p + 4 + UVp) + (size_t)n_recv * ((C + Co) * UVp + (size_t)C * Lo2p);
    return 256 + fl * sizeof(float) + (size_t)(n_recv + 1) * sizeof(int64_t) + 12 * 256;
}

// Projection problems of all degrees (l-dependent weights): one launch when the multi-problem kernel takes them, else
// `group` problems per launch (the factors / sectors of one degree).
static int launch_proj_degrees(const std::vector<ProjArgs>& v, int group, Kind kind, cudaStream_t st)
{
    if ((int)v.size() > group && get_math_mode() == CGTP_MATH_FP32 && !(kernel_path() & PATH_GENERIC_PROJ)) {
        bool handled = false;
        const int rc = launch_proj_multi(v.data(), (int)v.size(), kind, st, &handled);
        if (rc != CGTP_OK || handled) return rc;
    }
    for (size_t i = 0; i < v.size(); i += group) {
        const int n = (int)(v.size() - i) < group ? (int)(v.size() - i) : group;
        const int rc = launch_proj(&v[i], n, kind, st);
        if (rc) return rc;
    }
    return CGTP_OK;
}

// One run of the on-site pipeline S1-S5 over Ce even + Co odd rank channels (internal channel order: even block, then
// odd block).  cgtp_onsite is one pass; the parity-slot entry point (cgtp_onsite_parity) is four passes that differ in
// the input slots, the weight rows and the output sectors.
struct OnsitePass {
    const float *A, *B;   // first atom's [N, L2] block of each factor
    int64_t x_bs;         // floats between consecutive atoms
    const float *W_a, *W_b;
    const int* idx_in;    // [Ce+Co] device: row of W_a / W_b (row length N) of internal channel k
    const float* W_out;
    int ldw_out;          // floats between output rows n of W_out
    const int *idx_out_e, *idx_out_o;  // [Ce], [Co] device: offset of channel k inside a row of W_out
    int Ce, Co;
    float *out_e, *out_o; // first atom's [N, Lo2] block of the sector written by the even / odd channels
    int64_t o_bs;
    int accumulate;       // 1: add to the output sectors
    int sigma_C;          // 0: none; > 0: channel k keeps only the output degrees l with (l & 1) == ((k / sigma_C) & 1)
                          // inside its parity block (Eq.(54): (-1)^l = sigma)
    int64_t lw_in, lw_out;  // 0: l-shared weights; else floats between the weight matrices of consecutive degrees l
                          // (c_{cnl} of Eq.(35) :322, lambda_c^{(nl)} of Eq.(41) :346): S1 / S5 run once per degree
};

static int onsite_pass(const Plan* p, int N, const OnsitePass& q, int64_t batch, void* workspace, cudaStream_t st)
{
    const int Ce = q.Ce, Co = q.Co;
    // long steps (H of one factor beyond kPdlMaxBytes: configs[3] from lmax 12 up) launch their kernels in plain order
    PdlScope pdl((size_t)batch * (size_t)(Ce + Co) * p->L2 * sizeof(float) > kPdlMaxBytes);
    // the whole step in one kernel (onsite_fused.cu) when the shape fits and nothing but the plain contraction is asked
    if (!(kernel_path() & (PATH_UNFUSED_ONSITE | PATH_GENERIC_CORE | PATH_GENERIC_PROJ)) && get_math_mode() == CGTP_MATH_FP32 &&
        !q.lw_in && !q.lw_out && q.sigma_C == 0 && !q.accumulate && q.x_bs == (int64_t)N * p->L2 &&
        q.out_o == q.out_e + (size_t)N * p->Lo2 && q.o_bs == (int64_t)2 * N * p->Lo2) {
        bool handled = false;
        const int rc = launch_onsite_fused(p, N, Ce + Co, Ce, Co, q.A, q.B, q.W_a, q.W_b, q.idx_in, q.W_out, q.ldw_out,
                                           q.idx_out_e, q.idx_out_o, q.out_e, batch, st, &handled);
        if (rc != CGTP_OK || handled) return rc;
    }
    // fast core (onsite_core.cu) when both parities fit; it wants odd row strides and 32-column groups
    const bool fast = !(kernel_path() & PATH_GENERIC_CORE) && (Ce == 0 || onsite_fast_supported(p, false)) &&
                      (Co == 0 || onsite_fast_supported(p, true));
    const int hstr = fast ? onsite_fast_hstride(p) : p->L2p;
    const int tstr = fast ? onsite_fast_tstride(p) : p->Lo2p;
    const size_t ncol_e = (size_t)round_up((int)((size_t)batch * Ce % 32), 32) + (size_t)batch * Ce / 32 * 32;
    const size_t ncol_o = (size_t)round_up((int)((size_t)batch * Co % 32), 32) + (size_t)batch * Co / 32 * 32;

    Carver cv(workspace);
    float* Ha_e = cv.take<float>(ncol_e * hstr);
    float* Ha_o = cv.take<float>(ncol_o * hstr);
    float* Hb_e = cv.take<float>(ncol_e * hstr);
    float* Hb_o = cv.take<float>(ncol_o * hstr);
    float* T_e = cv.take<float>(ncol_e * tstr);
    float* T_o = cv.take<float>(ncol_o * tstr);
    if (fast) {
        // columns that pad the last group: define them (their results are never read)
        const size_t ne = (size_t)batch * Ce, no = (size_t)batch * Co;
        if (ncol_e > ne) {
            CGTP_CUDA_CHECK(cudaMemsetAsync(Ha_e + ne * hstr, 0, (ncol_e - ne) * hstr * 4, st));
            CGTP_CUDA_CHECK(cudaMemsetAsync(Hb_e + ne * hstr, 0, (ncol_e - ne) * hstr * 4, st));
        }
        if (ncol_o > no) {
            CGTP_CUDA_CHECK(cudaMemsetAsync(Ha_o + no * hstr, 0, (ncol_o - no) * hstr * 4, st));
            CGTP_CUDA_CHECK(cudaMemsetAsync(Hb_o + no * hstr, 0, (ncol_o - no) * hstr * 4, st));
        }
    }

    // S1: H = W . A (Eq.(35)); rows are written in parity-sorted channel order, even block then odd block.  With
    // l-dependent weights one launch per degree l over the columns l^2 .. l^2 + 2l of every row.
    int rc = CGTP_OK;
    std::vector<ProjArgs> pv;
    for (int l = 0; l < (q.lw_in ? p->lmax + 1 : 1); ++l) {
        for (int s = 0; s < 2; ++s) {
            pv.emplace_back();
            ProjArgs& a = pv.back();
            const int jo = q.lw_in ? l * l : 0;
            a.X = s ? q.B : q.A;
            a.x_bs = q.x_bs;
            a.x_rs = p->L2;
            a.W = (s ? q.W_b : q.W_a) + (size_t)l * q.lw_in;
            a.ldw_m = N;
            a.ldw_k = 1;
            a.idx_m = q.idx_in;
            a.idx_k = nullptr;
            a.M = Ce + Co;
            a.K = N;
            a.J = q.lw_in ? 2 * l + 1 : p->L2;
            a.out0 = (s ? Hb_e : Ha_e) + jo;
            a.o_bs0 = (int64_t)Ce * hstr;
            a.out1 = (s ? Hb_o : Ha_o) + jo;
            a.o_bs1 = (int64_t)Co * hstr;
            a.m_split = Ce;
            a.o_rs = hstr;
            a.batch = batch;
            a.accumulate = 0;
            a.j0 = jo;
        }
    }
    rc = launch_proj_degrees(pv, 2, K_PROJ_IN, st);
    if (rc) return rc;

    // S2-S4 fused, one launch per parity
    rc = fast ? launch_onsite_fast(p, false, Ha_e, Hb_e, T_e, batch * Ce, st)
              : launch_onsite_generic(p, false, Ha_e, Hb_e, T_e, batch * Ce, st);
    if (rc) return rc;
    rc = fast ? launch_onsite_fast(p, true, Ha_o, Hb_o, T_o, batch * Co, st)
              : launch_onsite_generic(p, true, Ha_o, Hb_o, T_o, batch * Co, st);
    if (rc) return rc;
    if (q.sigma_C > 0) {
        rc = launch_sigma_mask(T_e, tstr, batch * Ce, Ce, q.sigma_C, p->Lo2, st);
        if (rc) return rc;
        rc = launch_sigma_mask(T_o, tstr, batch * Co, Co, q.sigma_C, p->Lo2, st);
        if (rc) return rc;
    }

    // S5: out[b, s] = W_out[:, channels of sector s] . T_s (Eq.(41)); per degree with l-dependent weights
    pv.clear();
    for (int l = 0; l < (q.lw_out ? p->lmax_out + 1 : 1); ++l) {
        for (int s = 0; s < 2; ++s) {
            pv.emplace_back();
            ProjArgs& a = pv.back();
            const int jo = q.lw_out ? l * l : 0;
            a.X = s ? T_o : T_e;
            a.x_bs = (int64_t)(s ? Co : Ce) * tstr;
            a.x_rs = tstr;
            a.W = q.W_out + (size_t)l * q.lw_out;
            a.ldw_m = q.ldw_out;
            a.ldw_k = 1;
            a.idx_m = nullptr;
            a.idx_k = s ? q.idx_out_o : q.idx_out_e;
            a.M = N;
            a.K = s ? Co : Ce;
            a.J = q.lw_out ? 2 * l + 1 : p->Lo2;
            a.out0 = (s ? q.out_o : q.out_e) + jo;
            a.o_bs0 = q.o_bs;
            a.out1 = a.out0;
            a.o_bs1 = a.o_bs0;
            a.m_split = N;
            a.o_rs = p->Lo2;
            a.batch = batch;
            a.accumulate = q.accumulate;
            a.j0 = jo;
        }
    }
    return launch_proj_degrees(pv, 2, K_PROJ_OUT, st);
}

static int check_message_args(const float* node_feats, const int64_t* edge_index, const float* edge_vec,
                              const float* edge_radial, const float* W_node, const float* W_out, const float* out,
                              int64_t n_send, int64_t nodes, int64_t E, const void* workspace)
{
    if (nodes < 0 || n_send < 0 || E < 0) { set_error("negative size"); return CGTP_ERR_INVALID; }
    if (nodes == 0) return CGTP_OK;
    if (n_send == 0 && E > 0) { set_error("edges without sender nodes"); return CGTP_ERR_INVALID; }
    if ((!node_feats && n_send > 0) || !W_node || !W_out || !out || !workspace || (E > 0 && (!edge_index || !edge_vec || !edge_radial))) {
        set_error("null pointer argument");
        return CGTP_ERR_INVALID;
    }
    if (!aligned16(node_feats) || !aligned16(out) || !aligned16(W_node) || !aligned16(W_out) ||
        (E > 0 && (!aligned16(edge_index) || !aligned16(edge_vec) || !aligned16(edge_radial))) ||
        (reinterpret_cast<uintptr_t>(workspace) & 255u)) {
        set_error("misaligned pointer (tensors need 16-byte, workspace 256-byte alignment)");
        return CGTP_ERR_INVALID;
    }
    return CGTP_OK;
}

// One run of the message-passing pipeline M0-M6 over Ce even + Co odd rank channels; cgtp_message(_bipartite) is one
// pass, cgtp_message_parity two (one per source slot).
struct MessagePass {
    const float* node_feats;  // first sender's [N, L2] block
    int64_t x_bs;             // floats between consecutive senders
    const float* W_node;
    const int* idx_in;        // [Ce+Co] device: row of W_node (row length N) AND column of edge_radial of channel k
    const float* edge_radial;
    int radial_stride;        // floats between consecutive edges of edge_radial
    const float* W_out;
    int ldw_out;
    const int *idx_out_e, *idx_out_o;
    int Ce, Co;
    float *out_e, *out_o;
    int64_t o_bs;
    int accumulate;
    int sigma_C;              // as OnsitePass::sigma_C
    bool segments_done;       // row_ptr / status of this workspace are already built (second pass)
    int64_t lw_in, lw_out;    // as OnsitePass: l-dependent W_node (Eq.(47) :398) / W_out (Eq.(55), (58))
    bool radial_l1;           // edge_radial is [E][radial_stride][lmax+1]: l1-dependent R~ (Eq.(46) :396)
};

static int message_pass(const Plan* p, int N, const MessagePass& q, const int64_t* edge_index, const float* edge_vec,
                        int64_t n_send, int64_t nodes, int64_t E, void* workspace, cudaStream_t st)
{
    const int Ce = q.Ce, Co = q.Co;
    // long steps (node grids beyond kPdlMaxBytes: configs[4]) launch their kernels in plain order
    PdlScope pdl((size_t)n_send * (size_t)(Ce + Co) * p->UVp * sizeof(float) > kPdlMaxBytes);
    Carver cv(workspace);
    int32_t* status = cv.take<int32_t>(1);
    int64_t* row_ptr = cv.take<int64_t>((size_t)nodes + 1);
    const bool fast_synth = !(kernel_path() & PATH_GENERIC_SYNTH) && synth_fast_supported(p);
    const int hstr = fast_synth ? synth_fast_hstride(p) : p->L2p;
    float* H_e = cv.take<float>((size_t)round_up64(n_send * Ce, 32) * hstr);
    float* H_o = cv.take<float>((size_t)round_up64(n_send * Co, 32) * hstr);
    float* G_e = cv.take<float>((size_t)n_send * Ce * p->UVp);
    float* G_o = cv.take<float>((size_t)n_send * Co * p->UVp);
    float* S_e = cv.take<float>((size_t)nodes * Ce * p->UVp);
    float* S_o = cv.take<float>((size_t)nodes * Co * 2 * p->UVp);
    float* T_e = cv.take<float>((size_t)nodes * Ce * p->Lo2p);
    float* T_o = cv.take<float>((size_t)nodes * Co * p->Lo2p);

    // M0
    int rc = CGTP_OK;
    if (!q.segments_done) {
        rc = launch_segments(edge_index, E, nodes, n_send, row_ptr, status, st);
        if (rc) return rc;
    }

    // M1: H = W_node . node_feats (Eq.(47)); one launch per degree with l-dependent weights
    std::vector<ProjArgs> pv;
    for (int l = 0; l < (q.lw_in ? p->lmax + 1 : 1); ++l) {
        const int jo = q.lw_in ? l * l : 0;
        pv.emplace_back();
        ProjArgs& a = pv.back();
        a.X = q.node_feats;
        a.x_bs = q.x_bs;
        a.x_rs = p->L2;
        a.W = q.W_node + (size_t)l * q.lw_in;
        a.ldw_m = N;
        a.ldw_k = 1;
        a.idx_m = q.idx_in;
        a.idx_k = nullptr;
        a.M = Ce + Co;
        a.K = N;
        a.J = q.lw_in ? 2 * l + 1 : p->L2;
        a.out0 = H_e + jo;
        a.o_bs0 = (int64_t)Ce * hstr;
        a.out1 = H_o + jo;
        a.o_bs1 = (int64_t)Co * hstr;
        a.m_split = Ce;
        a.o_rs = hstr;
        a.batch = n_send;
        a.accumulate = 0;
        a.j0 = jo;
    }
    rc = launch_proj_degrees(pv, 1, K_PROJ_IN, st);
    if (rc) return rc;

    // M2 (value fields for both parities: the odd channels take their derivatives on the edge side and in M5)
    rc = fast_synth ? launch_node_synth_fast(p, false, H_e, hstr, G_e, n_send * Ce, st)
                    : launch_node_synth(p, false, H_e, G_e, n_send * Ce, st);
    if (rc) return rc;
    rc = fast_synth ? launch_node_synth_fast(p, true, H_o, hstr, G_o, n_send * Co, st)
                    : launch_node_synth(p, true, H_o, G_o, n_send * Co, st);
    if (rc) return rc;

    // M3 + M4
    if (q.radial_l1) {
        rc = launch_edge_lr(p, false, G_e, row_ptr, edge_index, E, edge_vec, q.edge_radial, q.idx_in, Ce, q.radial_stride, S_e, nodes, status, st);
        if (rc) return rc;
        rc = launch_edge_lr(p, true, G_o, row_ptr, edge_index, E, edge_vec, q.edge_radial, q.idx_in + Ce, Co, q.radial_stride, S_o, nodes, status, st);
        if (rc) return rc;
    } else {
        rc = launch_edge(p, false, G_e, row_ptr, edge_index, E, edge_vec, q.edge_radial, q.idx_in, Ce, q.radial_stride, S_e, nodes, status, st);
        if (rc) return rc;
        rc = launch_edge(p, true, G_o, row_ptr, edge_index, E, edge_vec, q.edge_radial, q.idx_in + Ce, Co, q.radial_stride, S_o, nodes, status, st);
        if (rc) return rc;
    }

    // M5
    rc = launch_analysis(p, false, S_e, T_e, nodes * Ce, st);
    if (rc) return rc;
    rc = launch_analysis(p, true, S_o, T_o, nodes * Co, st);
    if (rc) return rc;
    if (q.sigma_C > 0) {
        rc = launch_sigma_mask(T_e, p->Lo2p, nodes * Ce, Ce, q.sigma_C, p->Lo2, st);
        if (rc) return rc;
        rc = launch_sigma_mask(T_o, p->Lo2p, nodes * Co, Co, q.sigma_C, p->Lo2, st);
        if (rc) return rc;
    }

    // M6 (per degree with l-dependent weights)
    pv.clear();
    for (int l = 0; l < (q.lw_out ? p->lmax_out + 1 : 1); ++l) {
        const int jo = q.lw_out ? l * l : 0;
        for (int s = 0; s < 2; ++s) {
            pv.emplace_back();
            ProjArgs& b = pv.back();
            b.X = s ? T_o : T_e;
            b.x_bs = (int64_t)(s ? Co : Ce) * p->Lo2p;
            b.x_rs = p->Lo2p;
            b.W = q.W_out + (size_t)l * q.lw_out;
            b.ldw_m = q.ldw_out;
            b.ldw_k = 1;
            b.idx_m = nullptr;
            b.idx_k = s ? q.idx_out_o : q.idx_out_e;
            b.M = N;
            b.K = s ? Co : Ce;
            b.J = q.lw_out ? 2 * l + 1 : p->Lo2;
            b.out0 = (s ? q.out_o : q.out_e) + jo;
            b.o_bs0 = q.o_bs;
            b.out1 = b.out0;
            b.o_bs1 = b.o_bs0;
            b.m_split = N;
            b.o_rs = p->Lo2;
            b.batch = nodes;
            b.accumulate = q.accumulate;
            b.j0 = jo;
        }
    }
    return launch_proj_degrees(pv, 2, K_PROJ_OUT, st);
}

}  // namespace cgtp

using namespace cgtp;

extern "C" {

int cgtp_version(void) { return 100; }
const char* cgtp_last_error(void) { return cgtp::last_error(); }
int cgtp_max_lmax(void) { return kMaxBand; }

int cgtp_grid_shape(int lmax, int lmax_out, int* U, int* V)
{
    if (lmax < 0 || lmax_out < 0 || lmax_out > 2 * lmax) { set_error("invalid band limits"); return CGTP_ERR_INVALID; }
    if (U) *U = (2 * lmax + lmax_out + 2) / 2;
    if (V) *V = 2 * lmax + lmax_out + 1;
    return CGTP_OK;
}

int cgtp_grid_shape_nu(int lmax, int lmax_out, int nu, int* U, int* V)
{
    if (nu < 1 || lmax < 0 || lmax_out < 0 || (int64_t)lmax_out > (int64_t)nu * lmax) {
        set_error("invalid band limits / body order");
        return CGTP_ERR_INVALID;
    }
    if (U) *U = (nu * lmax + lmax_out + 2) / 2;
    if (V) *V = nu * lmax + lmax_out + 1;
    return CGTP_OK;
}

size_t cgtp_onsite_workspace_bytes(int lmax, int lmax_out, int N, int C, int64_t batch)
{
    (void)N;
    if (lmax < 0 || lmax_out < 0 || C <= 0 || batch < 0) return 0;
    return onsite_ws_bytes(lmax, lmax_out, C, batch);
}

static int onsite_entry(bool lw, const float* A, const float* B, const float* W_a, const float* W_b, const float* W_out,
                        int lmax, int lmax_out, int N, int C, const uint8_t* parity_mask, float* out, int64_t batch,
                        void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    clear_error();
    int rc = check_common(lmax, lmax_out, N, C, parity_mask);
    if (rc) return rc;
    if (batch < 0) { set_error("negative batch"); return CGTP_ERR_INVALID; }
    if (batch == 0) return CGTP_OK;
    if (!A || !B || !W_a || !W_b || !W_out || !out || !workspace) { set_error("null pointer argument"); return CGTP_ERR_INVALID; }
    if (!aligned16(A) || !aligned16(B) || !aligned16(out) || !aligned16(W_a) || !aligned16(W_b) || !aligned16(W_out) ||
        (reinterpret_cast<uintptr_t>(workspace) & 255u)) {
        set_error("misaligned pointer (tensors need 16-byte, workspace 256-byte alignment)");
        return CGTP_ERR_INVALID;
    }
    if (workspace_bytes < onsite_ws_bytes(lmax, lmax_out, C, batch)) {
        set_error("workspace too small: %zu < %zu bytes", workspace_bytes, onsite_ws_bytes(lmax, lmax_out, C, batch));
        return CGTP_ERR_INVALID;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const Plan* p = get_plan(lmax, lmax_out);
    if (!p) return CGTP_ERR_CUDA;
    const ChannelPlan* cp = get_channel_plan(C, parity_mask);
    if (!cp) return CGTP_ERR_CUDA;
    OnsitePass q;
    q.A = A;
    q.B = B;
    q.x_bs = (int64_t)N * p->L2;
    q.W_a = W_a;
    q.W_b = W_b;
    q.idx_in = cp->perm_dev;
    q.W_out = W_out;
    q.ldw_out = C;
    q.idx_out_e = cp->perm_dev;
    q.idx_out_o = cp->perm_dev + cp->Ce;
    q.Ce = cp->Ce;
    q.Co = cp->Co;
    q.out_e = out;
    q.out_o = out + (size_t)N * p->Lo2;
    q.o_bs = (int64_t)2 * N * p->Lo2;
    q.accumulate = 0;
    q.sigma_C = 0;
    q.lw_in = lw ? (int64_t)C * N : 0;
    q.lw_out = lw ? (int64_t)N * C : 0;
    return onsite_pass(p, N, q, batch, workspace, st);
}

size_t cgtp_message_workspace_bytes(int lmax, int lmax_out, int N, int C, const uint8_t* parity_mask, int64_t nodes,
                                    int64_t E)
{
    (void)N;
    (void)E;
    if (lmax < 0 || lmax_out < 0 || C <= 0 || nodes < 0 || !parity_mask) return 0;
    int Co = 0;
    for (int c = 0; c < C; ++c) Co += parity_mask[c] ? 1 : 0;
    return message_ws_bytes(lmax, lmax_out, C, Co, nodes, nodes);
}

size_t cgtp_message_bipartite_workspace_bytes(int lmax, int lmax_out, int N, int C, const uint8_t* parity_mask,
                                              int64_t n_send, int64_t n_recv, int64_t E)
{
    (void)N;
    (void)E;
    if (lmax < 0 || lmax_out < 0 || C <= 0 || n_send < 0 || n_recv < 0 || !parity_mask) return 0;
    int Co = 0;
    for (int c = 0; c < C; ++c) Co += parity_mask[c] ? 1 : 0;
    return message_ws_bytes(lmax, lmax_out, C, Co, n_send, n_recv);
}

int cgtp_build_segments(const int64_t* edge_index, int64_t E, int64_t nodes, int64_t* row_ptr, int32_t* status,
                        void* cuda_stream)
{
    clear_error();
    if (E < 0 || nodes < 0) { set_error("negative size"); return CGTP_ERR_INVALID; }
    if ((!edge_index && E > 0) || !row_ptr || !status) { set_error("null pointer argument"); return CGTP_ERR_INVALID; }
    return launch_segments(edge_index, E, nodes, nodes, row_ptr, status, static_cast<cudaStream_t>(cuda_stream));
}

static int message_entry(int lw, const float* node_feats, const int64_t* edge_index, const float* edge_vec,
                         const float* edge_radial, const float* W_node, const float* W_out, int lmax, int lmax_out,
                         int N, int C, const uint8_t* parity_mask, float* out, int64_t n_send, int64_t nodes,
                         int64_t E, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    clear_error();
    int rc = check_common(lmax, lmax_out, N, C, parity_mask);
    if (rc) return rc;
    rc = check_message_args(node_feats, edge_index, edge_vec, edge_radial, W_node, W_out, out, n_send, nodes, E, workspace);
    if (rc || nodes == 0) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const Plan* p = get_plan(lmax, lmax_out);
    if (!p) return CGTP_ERR_CUDA;
    const ChannelPlan* cp = get_channel_plan(C, parity_mask);
    if (!cp) return CGTP_ERR_CUDA;
    const int Ce = cp->Ce, Co = cp->Co;
    if (workspace_bytes < message_ws_bytes(lmax, lmax_out, C, Co, n_send, nodes)) {
        set_error("workspace too small: %zu < %zu bytes", workspace_bytes, message_ws_bytes(lmax, lmax_out, C, Co, n_send, nodes));
        return CGTP_ERR_INVALID;
    }
    MessagePass q;
    q.node_feats = node_feats;
    q.x_bs = (int64_t)N * p->L2;
    q.W_node = W_node;
    q.idx_in = cp->perm_dev;
    q.edge_radial = edge_radial;
    q.radial_stride = C;
    q.W_out = W_out;
    q.ldw_out = C;
    q.idx_out_e = cp->perm_dev;
    q.idx_out_o = cp->perm_dev + Ce;
    q.Ce = Ce;
    q.Co = Co;
    q.out_e = out;
    q.out_o = out + (size_t)N * p->Lo2;
    q.o_bs = (int64_t)2 * N * p->Lo2;
    q.accumulate = 0;
    q.sigma_C = 0;
    q.segments_done = false;
    q.lw_in = lw ? (int64_t)C * N : 0;
    q.lw_out = lw ? (int64_t)N * C : 0;
    q.radial_l1 = lw == 2;
    return message_pass(p, N, q, edge_index, edge_vec, n_send, nodes, E, workspace, st);
}

int cgtp_onsite(const float* A, const float* B, const float* W_a, const float* W_b, const float* W_out, int lmax,
                int lmax_out, int N, int C, const uint8_t* parity_mask, float* out, int64_t batch, void* workspace,
                size_t workspace_bytes, void* cuda_stream)
{
    return onsite_entry(false, A, B, W_a, W_b, W_out, lmax, lmax_out, N, C, parity_mask, out, batch, workspace,
                        workspace_bytes, cuda_stream);
}

int cgtp_onsite_lw(const float* A, const float* B, const float* W_a, const float* W_b, const float* W_out, int lmax,
                   int lmax_out, int N, int C, const uint8_t* parity_mask, float* out, int64_t batch, void* workspace,
                   size_t workspace_bytes, void* cuda_stream)
{
    return onsite_entry(true, A, B, W_a, W_b, W_out, lmax, lmax_out, N, C, parity_mask, out, batch, workspace,
                        workspace_bytes, cuda_stream);
}

int cgtp_message_bipartite(const float* node_feats, const int64_t* edge_index, const float* edge_vec,
                           const float* edge_radial, const float* W_node, const float* W_out, int lmax, int lmax_out,
                           int N, int C, const uint8_t* parity_mask, float* out, int64_t n_send, int64_t nodes,
                           int64_t E, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    return message_entry(0, node_feats, edge_index, edge_vec, edge_radial, W_node, W_out, lmax, lmax_out, N, C,
                         parity_mask, out, n_send, nodes, E, workspace, workspace_bytes, cuda_stream);
}

int cgtp_message_lw(const float* node_feats, const int64_t* edge_index, const float* edge_vec, const float* edge_radial,
                    const float* W_node, const float* W_out, int lmax, int lmax_out, int N, int C,
                    const uint8_t* parity_mask, float* out, int64_t nodes, int64_t E, void* workspace,
                    size_t workspace_bytes, void* cuda_stream)
{
    return message_entry(1, node_feats, edge_index, edge_vec, edge_radial, W_node, W_out, lmax, lmax_out, N, C,
                         parity_mask, out, nodes, nodes, E, workspace, workspace_bytes, cuda_stream);
}

int cgtp_message_lwr(const float* node_feats, const int64_t* edge_index, const float* edge_vec, const float* edge_radial,
                     const float* W_node, const float* W_out, int lmax, int lmax_out, int N, int C,
                     const uint8_t* parity_mask, float* out, int64_t nodes, int64_t E, void* workspace,
                     size_t workspace_bytes, void* cuda_stream)
{
    return message_entry(2, node_feats, edge_index, edge_vec, edge_radial, W_node, W_out, lmax, lmax_out, N, C,
                         parity_mask, out, nodes, nodes, E, workspace, workspace_bytes, cuda_stream);
}

int cgtp_message(const float* node_feats, const int64_t* edge_index, const float* edge_vec, const float* edge_radial,
                 const float* W_node, const float* W_out, int lmax, int lmax_out, int N, int C,
                 const uint8_t* parity_mask, float* out, int64_t nodes, int64_t E, void* workspace,
                 size_t workspace_bytes, void* cuda_stream)
{
    return cgtp_message_bipartite(node_feats, edge_index, edge_vec, edge_radial, W_node, W_out, lmax, lmax_out, N, C,
                                  parity_mask, out, nodes, nodes, E, workspace, workspace_bytes, cuda_stream);
}

int cgtp_message_status(const void* workspace, void* cuda_stream)
{
    clear_error();
    if (!workspace) { set_error("null workspace"); return CGTP_ERR_INVALID; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    CGTP_CUDA_CHECK(cudaStreamSynchronize(st));
    int32_t h = 0;
    CGTP_CUDA_CHECK(cudaMemcpy(&h, workspace, sizeof h, cudaMemcpyDeviceToHost));
    if (h != 0) {
        set_error("edge_index is not receiver-sorted or has an index outside [0, nodes)");
        return CGTP_ERR_GRAPH;
    }
    return CGTP_OK;
}

// ------------------------------------------------------------------------------ nu-body on-site product
static size_t nbody_ws_bytes(int nu, int lmax, int lmax_out, int C, int64_t batch)
{
    const size_t L2p = round_up((lmax + 1) * (lmax + 1), 4), Lo2p = round_up((lmax_out + 1) * (lmax_out + 1), 4);
    // H rows have the odd stride L2 | 1 <= L2p + 1; every factor block is padded to whole groups of 4 columns (nu = 2
    // runs on the bilinear core: groups of 32 columns, T rows of stride Lo2 | 1)
    return (((size_t)batch * C + 32) * (size_t)nu * (L2p + 1) + 4 * (L2p + 1) + ((size_t)batch * C + 32) * (Lo2p + 1)) * sizeof(float) +
           4 * 256;
}

size_t cgtp_onsite_nbody_workspace_bytes(int nu, int lmax, int lmax_out, int N, int C, int64_t batch)
{
    (void)N;
    if (nu < 1 || lmax < 0 || lmax_out < 0 || C <= 0 || batch < 0) return 0;
    return nbody_ws_bytes(nu, lmax, lmax_out, C, batch);
}

int cgtp_onsite_nbody(const float* X, const float* W_in, const float* W_out, int nu, int lmax, int lmax_out, int N,
                      int C, float* out, int64_t batch, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    clear_error();
    if (nu < 1) { set_error("body order nu=%d must be >= 1", nu); return CGTP_ERR_INVALID; }
    if (lmax < 0 || lmax_out < 0 || (int64_t)lmax_out > (int64_t)nu * lmax) {
        set_error("invalid band limits lmax=%d lmax_out=%d (need 0 <= lmax_out <= nu*lmax)", lmax, lmax_out);
        return CGTP_ERR_INVALID;
    }
    if (N <= 0 || C <= 0) { set_error("N and C must be positive (N=%d, C=%d)", N, C); return CGTP_ERR_INVALID; }
    const int LB = kernel_band(lmax > lmax_out ? lmax : lmax_out);
    if (!nbody_supported(LB, nu)) {
        set_error("nu-body product: max(lmax,lmax_out)=%d / nu=%d exceed the compiled limits (band limit 20, nu 4)",
                  lmax > lmax_out ? lmax : lmax_out, nu);
        return CGTP_ERR_UNSUPPORTED;
    }
    if (batch < 0) { set_error("negative batch"); return CGTP_ERR_INVALID; }
    if (batch == 0) return CGTP_OK;
    if (!X || !W_in || !W_out || !out || !workspace) { set_error("null pointer argument"); return CGTP_ERR_INVALID; }
    if (!aligned16(X) || !aligned16(out) || !aligned16(W_in) || !aligned16(W_out) ||
        (reinterpret_cast<uintptr_t>(workspace) & 255u)) {
        set_error("misaligned pointer (tensors need 16-byte, workspace 256-byte alignment)");
        return CGTP_ERR_INVALID;
    }
    if (workspace_bytes < nbody_ws_bytes(nu, lmax, lmax_out, C, batch)) {
        set_error("workspace too small: %zu < %zu bytes", workspace_bytes, nbody_ws_bytes(nu, lmax, lmax_out, C, batch));
        return CGTP_ERR_INVALID;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const Plan* p = get_plan_nu(lmax, lmax_out, nu);
    if (!p) return CGTP_ERR_CUDA;
    const int64_t ncols = batch * C;
    PdlScope pdl((size_t)ncols * p->L2 * sizeof(float) > kPdlMaxBytes);  // long steps: plain launch order (common.cuh)
    Carver cv(workspace);
    const int hstr = nbody_hstride(p);
    // nu = 2 is the pointwise product of the bilinear step (Eq.(38) PAPER.md:332 with every channel even): the bilinear
    // core runs it (H blocks padded to groups of 32 columns, T rows of its odd stride)
    const Plan* p2 = (nu == 2 && !(kernel_path() & PATH_GENERIC_CORE)) ? get_plan(lmax, lmax_out) : nullptr;
    const bool bilinear = p2 && onsite_fast_supported(p2, false) && onsite_fast_hstride(p2) == hstr;
    // nu >= 3 at small band limits: one thread per column (nbody_reg.cu), same padded layout
    const bool regcore = !bilinear && !(kernel_path() & PATH_SMEM_CORE) && nbody_reg_supported(p);
    const bool pad32 = bilinear || regcore;
    const int64_t hfs = pad32 ? (int64_t)round_up64(ncols, 32) * hstr : nbody_hfstride(p, ncols);
    const int tstr = pad32 ? (p->Lo2 | 1) : p->Lo2p;
    float* H = cv.take<float>((size_t)nu * hfs + 4 * hstr);
    float* T = cv.take<float>((size_t)(pad32 ? round_up64(ncols, 32) : ncols) * tstr);

    // S1 per factor: H[s] = W_in[s] . X[s] (Eq.(35)), one launch over the nu problems
    std::vector<ProjArgs> pv(nu);
    for (int s = 0; s < nu; ++s) {
        ProjArgs& a = pv[s];
        a.X = X + (size_t)s * batch * N * p->L2;
        a.x_bs = (int64_t)N * p->L2;
        a.x_rs = p->L2;
        a.W = W_in + (size_t)s * C * N;
        a.ldw_m = N;
        a.ldw_k = 1;
        a.idx_m = nullptr;
        a.idx_k = nullptr;
        a.M = C;
        a.K = N;
        a.J = p->L2;
        a.out0 = H + (size_t)s * hfs;
        a.o_bs0 = (int64_t)C * hstr;
        a.out1 = a.out0;
        a.o_bs1 = a.o_bs0;
        a.m_split = C;
        a.o_rs = hstr;
        a.batch = batch;
        a.accumulate = 0;
        a.j0 = 0;
    }
    int rc = launch_proj_degrees(pv, 2, K_PROJ_IN, st);
    if (rc) return rc;
    // S2-S4 with nu factors
    rc = bilinear  ? launch_onsite_fast(p2, false, H, H + hfs, T, round_up64(ncols, 32), st)
         : regcore ? launch_nbody_reg(p, H, hfs, T, ncols, st)
                   : launch_nbody(p, H, T, ncols, st);
    if (rc) return rc;
    // S5: out[b] = W_out . T[b] (Eq.(41) :346)
    std::vector<ProjArgs> po(1);
    {
        ProjArgs& a = po[0];
        a.X = T;
        a.x_bs = (int64_t)C * tstr;
        a.x_rs = tstr;
        a.W = W_out;
        a.ldw_m = C;
        a.ldw_k = 1;
        a.idx_m = nullptr;
        a.idx_k = nullptr;
        a.M = N;
        a.K = C;
        a.J = p->Lo2;
        a.out0 = out;
        a.o_bs0 = (int64_t)N * p->Lo2;
        a.out1 = a.out0;
        a.o_bs1 = a.o_bs0;
        a.m_split = N;
        a.o_rs = p->Lo2;
        a.batch = batch;
        a.accumulate = 0;
        a.j0 = 0;
    }
    return launch_proj_degrees(po, 1, K_PROJ_OUT, st);
}

// ------------------------------------------------------------------------------ two feature fields, Eq.(28)
// Edges are processed in chunks of at most field_chunk(C) so that the per-edge buffers stay bounded (<= 2^22 columns).
static int64_t field_chunk(int C, int64_t E)
{
    const int64_t cap = ((int64_t)1 << 22) / C;
    return E < cap ? E : cap;
}

static size_t field_ws_bytes(int lmax, int lmax_out, int C, int64_t n_send, int64_t nodes, int64_t E)
{
    const size_t L2p = round_up((lmax + 1) * (lmax + 1), 4), Lo2p = round_up((lmax_out + 1) * (lmax_out + 1), 4);
    const size_t ec = (size_t)field_chunk(C, E);
    // per chunk: Ha, Hb (two parities, columns padded to groups of 32), T; per node: Hn, Tn; status, row_ptr
    const size_t fl = (ec * C + 128) * (2 * (L2p + 4) + (Lo2p + 4)) + ((size_t)n_send * C + 128) * (L2p + 4) +
                      ((size_t)nodes * C + 128) * (Lo2p + 4);
    return 256 + fl * sizeof(float) + (size_t)(nodes + 1) * sizeof(int64_t) + 16 * 256;
}

size_t cgtp_message_field_bipartite_workspace_bytes(int lmax, int lmax_out, int N, int Ne, int C, int64_t n_send,
                                                    int64_t nodes, int64_t E)
{
    (void)N;
    (void)Ne;
    if (lmax < 0 || lmax_out < 0 || C <= 0 || n_send < 0 || nodes < 0 || E < 0) return 0;
    return field_ws_bytes(lmax, lmax_out, C, n_send, nodes, E);
}

size_t cgtp_message_field_workspace_bytes(int lmax, int lmax_out, int N, int Ne, int C, int64_t nodes, int64_t E)
{
    return cgtp_message_field_bipartite_workspace_bytes(lmax, lmax_out, N, Ne, C, nodes, nodes, E);
}

// lw: l-dependent weights W_edge [lmax+1, C, Ne], W_node [lmax+1, C, N], W_out [lmax_out+1, N, C] (Eq.(35), (41), (47), (55)):
// every projection becomes one problem per degree l over the columns l^2 .. l^2 + 2l (one launch with proj_multi).
// One run of the two-field pipeline (Eq.(28)) over Ce even + Co odd rank channels; cgtp_message_field is one
// pass, cgtp_message_field_parity four (one per pair of input slots).
struct FieldPass {
    const float* node_feats;  // first sender's [N, L2] block
    int64_t x_bs_node;        // floats between consecutive senders
    const float* edge_feats;  // first edge's [Ne, L2] block
    int64_t x_bs_edge;        // floats between consecutive edges
    const float *W_edge, *W_node;
    const int* idx_in;        // [Ce+Co] device: row of W_edge (row length Ne) and of W_node (row length N) of channel k
    const float* W_out;
    int ldw_out;
    const int *idx_out_e, *idx_out_o;
    int Ce, Co;
    float *out_e, *out_o;
    int64_t o_bs;
    int accumulate;
    int sigma_C;              // as OnsitePass::sigma_C
    bool segments_done;
    bool lw;
};

static int field_pass(const Plan* p, int N, int Ne, const FieldPass& q, const int64_t* edge_index, int64_t n_send,
                      int64_t nodes, int64_t E, void* workspace, cudaStream_t st)
{
    const int C = q.Ce + q.Co;
    const int Cpar[2] = {q.Ce, q.Co};
    const bool lw = q.lw;
    int rc = CGTP_OK;
    PdlScope pdl((size_t)E * (size_t)C * p->L2 * sizeof(float) > kPdlMaxBytes);  // long steps: plain launch order (common.cuh)
    const bool fast = !(kernel_path() & PATH_GENERIC_CORE) && (Cpar[0] == 0 || onsite_fast_supported(p, false)) &&
                      (Cpar[1] == 0 || onsite_fast_supported(p, true));
    const int hstr = fast ? onsite_fast_hstride(p) : p->L2p;
    const int tstr = fast ? onsite_fast_tstride(p) : p->Lo2p;
    const int64_t ec_max = field_chunk(C, E);

    Carver cv(workspace);
    int32_t* status = cv.take<int32_t>(1);
    int64_t* row_ptr = cv.take<int64_t>((size_t)nodes + 1);
    float *Hn[2], *Tn[2], *Ha[2], *Hb[2], *T[2];
    size_t ncol[2];
    for (int s = 0; s < 2; ++s) {
        ncol[s] = (size_t)round_up64(ec_max * Cpar[s], 32);
        Hn[s] = cv.take<float>((size_t)n_send * Cpar[s] * hstr);
        Tn[s] = cv.take<float>((size_t)nodes * Cpar[s] * tstr);
        Ha[s] = cv.take<float>(ncol[s] * hstr);
        Hb[s] = cv.take<float>(ncol[s] * hstr);
        T[s] = cv.take<float>(ncol[s] * tstr);
    }

    // M0
    if (!q.segments_done) {
        rc = launch_segments(edge_index, E, nodes, n_send, row_ptr, status, st);
        if (rc) return rc;
    }
    // the pool kernel leaves Tn alone when M0 flags the edge list: define it, so that `out` is zeros plus the flag
    for (int s = 0; s < 2; ++s)
        if (Cpar[s] > 0 && nodes > 0) CGTP_CUDA_CHECK(cudaMemsetAsync(Tn[s], 0, (size_t)nodes * Cpar[s] * tstr * 4, st));

    // factor 2: Hn = W_node . node_feats, once per node (Eq.(47) :398)
    ProjArgs a;
    a.X = q.node_feats;
    a.x_bs = q.x_bs_node;
    a.x_rs = p->L2;
    a.W = q.W_node;
    a.ldw_m = N;
    a.ldw_k = 1;
    a.idx_m = q.idx_in;
    a.idx_k = nullptr;
    a.M = C;
    a.K = N;
    a.J = p->L2;
    a.out0 = Hn[0];
    a.o_bs0 = (int64_t)Cpar[0] * hstr;
    a.out1 = Hn[1];
    a.o_bs1 = (int64_t)Cpar[1] * hstr;
    a.m_split = Cpar[0];
    a.o_rs = hstr;
    a.batch = n_send;
    a.accumulate = 0;
    a.j0 = 0;
    // one problem per degree with l-dependent weights, else the whole row
    auto per_degree = [&](const ProjArgs& base, const float* W, int K) {
        std::vector<ProjArgs> v;
        for (int l = 0; l < (lw ? p->lmax + 1 : 1); ++l) {
            ProjArgs d = base;
            const int jo = lw ? l * l : 0;
            d.W = W + (lw ? (size_t)l * C * K : 0);
            d.J = lw ? 2 * l + 1 : p->L2;
            d.out0 = base.out0 + jo;
            d.out1 = base.out1 + jo;
            d.j0 = jo;
            v.push_back(d);
        }
        return v;
    };
    if (n_send > 0) {
        rc = launch_proj_degrees(per_degree(a, q.W_node, N), 1, K_PROJ_IN, st);
        if (rc) return rc;
    }

    for (int64_t e0 = 0; e0 == 0 || e0 < E; e0 += ec_max) {
        const int64_t ec = E - e0 < ec_max ? E - e0 : ec_max;
        if (ec > 0) {
            // factor 1: Ha = W_edge . edge_feats ("an explicit radial contraction ... on the edge side", :471)
            ProjArgs b = a;
            b.X = q.edge_feats + (size_t)e0 * q.x_bs_edge;
            b.x_bs = q.x_bs_edge;
            b.W = q.W_edge;
            b.ldw_m = Ne;
            b.K = Ne;
            b.out0 = Ha[0];
            b.out1 = Ha[1];
            b.batch = ec;
            rc = launch_proj_degrees(per_degree(b, q.W_edge, Ne), 1, K_PROJ_IN, st);
            if (rc) return rc;
        }
        for (int s = 0; s < 2; ++s) {
            const int64_t nc = ec * Cpar[s];
            if (nc > 0 && fast && !(kernel_path() & PATH_FIELD_PER_EDGE)) {
                // neighbour sum on the grid inside the core (Eq.(52) :415): one inverse transform and one analysis per
                // receiver, nothing per edge written to HBM
                bool pooled = false;
                rc = launch_field_pool_core(p, s == 1, Ha[s], Hn[s], edge_index, row_ptr, Cpar[s], status, Tn[s], nodes, e0,
                                            e0 + ec, st, &pooled);
                if (rc) return rc;
                if (pooled) continue;
            }
            if (nc > 0) {
                // S2-S4 per edge: the edge field is factor 1 (R10), the sender's field factor 2 -- read in place through
                // the edge list when the core's column groups do not straddle edges, else gathered into Hb first
                bool handled = false;
                if (fast) {
                    rc = launch_onsite_fast_gather(p, s == 1, Ha[s], Hn[s], edge_index + e0, Cpar[s], status, T[s], nc, st,
                                                   &handled);
                    if (rc) return rc;
                }
                if (!handled) {
                    const size_t pad = (size_t)round_up64(nc, 32) - (size_t)nc;
                    if (pad) {  // columns that pad the last group of 32: defined, never read back
                        CGTP_CUDA_CHECK(cudaMemsetAsync(Ha[s] + (size_t)nc * hstr, 0, pad * hstr * 4, st));
                        CGTP_CUDA_CHECK(cudaMemsetAsync(Hb[s] + (size_t)nc * hstr, 0, pad * hstr * 4, st));
                    }
                    rc = launch_field_gather(Hn[s], edge_index + e0, Hb[s], ec, Cpar[s] * hstr, status, st);
                    if (rc) return rc;
                    rc = fast ? launch_onsite_fast(p, s == 1, Ha[s], Hb[s], T[s], nc, st)
                              : launch_onsite_generic(p, s == 1, Ha[s], Hb[s], T[s], nc, st);
                    if (rc) return rc;
                }
            }
            // sum over the in-edges of every receiver (Eq.(28) sum_j), in edge order
            if (Cpar[s] > 0) {
                rc = launch_field_pool(T[s], row_ptr, Tn[s], nodes, e0, e0 + ec, Cpar[s] * tstr, status, st);
                if (rc) return rc;
            }
        }
        if (E == 0) break;
    }

    if (q.sigma_C > 0)
        for (int s = 0; s < 2; ++s)
            if (Cpar[s] > 0) {
                rc = launch_sigma_mask(Tn[s], tstr, nodes * Cpar[s], Cpar[s], q.sigma_C, p->Lo2, st);
                if (rc) return rc;
            }

    // output projection per receiver (Eq.(55), (58))
    std::vector<ProjArgs> pv;
    for (int l = 0; l < (lw ? p->lmax_out + 1 : 1); ++l) {
        const int jo = lw ? l * l : 0;
        for (int s = 0; s < 2; ++s) {
            pv.emplace_back();
            ProjArgs& o = pv.back();
            o.X = Tn[s];
            o.x_bs = (int64_t)Cpar[s] * tstr;
            o.x_rs = tstr;
            o.W = q.W_out + (lw ? (size_t)l * N * C : 0);
            o.ldw_m = q.ldw_out;
            o.ldw_k = 1;
            o.idx_m = nullptr;
            o.idx_k = s ? q.idx_out_o : q.idx_out_e;
            o.M = N;
            o.K = Cpar[s];
            o.J = lw ? 2 * l + 1 : p->Lo2;
            o.out0 = (s ? q.out_o : q.out_e) + jo;
            o.o_bs0 = q.o_bs;
            o.out1 = o.out0;
            o.o_bs1 = o.o_bs0;
            o.m_split = N;
            o.o_rs = p->Lo2;
            o.batch = nodes;
            o.accumulate = q.accumulate;
            o.j0 = jo;
        }
    }
    return launch_proj_degrees(pv, 2, K_PROJ_OUT, st);
}


static int field_entry(bool lw, const float* node_feats, const int64_t* edge_index, const float* edge_feats,
                       const float* W_edge, const float* W_node, const float* W_out, int lmax, int lmax_out, int N, int Ne,
                       int C, const uint8_t* parity_mask, float* out, int64_t n_send, int64_t nodes, int64_t E,
                       void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    clear_error();
    int rc = check_common(lmax, lmax_out, N, C, parity_mask);
    if (rc) return rc;
    if (Ne <= 0) { set_error("Ne must be positive (Ne=%d)", Ne); return CGTP_ERR_INVALID; }
    if (nodes < 0 || n_send < 0 || E < 0) { set_error("negative size"); return CGTP_ERR_INVALID; }
    if (nodes == 0) return CGTP_OK;
    if (n_send == 0 && E > 0) { set_error("edges without sender nodes"); return CGTP_ERR_INVALID; }
    if ((!node_feats && n_send > 0) || !W_edge || !W_node || !W_out || !out || !workspace || (E > 0 && (!edge_index || !edge_feats))) {
        set_error("null pointer argument");
        return CGTP_ERR_INVALID;
    }
    if (!aligned16(node_feats) || !aligned16(out) || !aligned16(W_edge) || !aligned16(W_node) || !aligned16(W_out) ||
        (E > 0 && (!aligned16(edge_index) || !aligned16(edge_feats))) || (reinterpret_cast<uintptr_t>(workspace) & 255u)) {
        set_error("misaligned pointer (tensors need 16-byte, workspace 256-byte alignment)");
        return CGTP_ERR_INVALID;
    }
    if (workspace_bytes < field_ws_bytes(lmax, lmax_out, C, n_send, nodes, E)) {
        set_error("workspace too small: %zu < %zu bytes", workspace_bytes, field_ws_bytes(lmax, lmax_out, C, n_send, nodes, E));
        return CGTP_ERR_INVALID;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const Plan* p = get_plan(lmax, lmax_out);
    if (!p) return CGTP_ERR_CUDA;
    const ChannelPlan* cp = get_channel_plan(C, parity_mask);
    if (!cp) return CGTP_ERR_CUDA;
    FieldPass q;
    q.node_feats = node_feats;
    q.x_bs_node = (int64_t)N * p->L2;
    q.edge_feats = edge_feats;
    q.x_bs_edge = (int64_t)Ne * p->L2;
    q.W_edge = W_edge;
    q.W_node = W_node;
    q.idx_in = cp->perm_dev;
    q.W_out = W_out;
    q.ldw_out = C;
    q.idx_out_e = cp->perm_dev;
    q.idx_out_o = cp->perm_dev + cp->Ce;
    q.Ce = cp->Ce;
    q.Co = cp->Co;
    q.out_e = out;
    q.out_o = out + (size_t)N * p->Lo2;
    q.o_bs = (int64_t)2 * N * p->Lo2;
    q.accumulate = 0;
    q.sigma_C = 0;
    q.segments_done = false;
    q.lw = lw;
    return field_pass(p, N, Ne, q, edge_index, n_send, nodes, E, workspace, st);
}

int cgtp_message_field(const float* node_feats, const int64_t* edge_index, const float* edge_feats, const float* W_edge,
                       const float* W_node, const float* W_out, int lmax, int lmax_out, int N, int Ne, int C,
                       const uint8_t* parity_mask, float* out, int64_t nodes, int64_t E, void* workspace,
                       size_t workspace_bytes, void* cuda_stream)
{
    return cgtp_message_field_bipartite(node_feats, edge_index, edge_feats, W_edge, W_node, W_out, lmax, lmax_out, N, Ne, C,
                                        parity_mask, out, nodes, nodes, E, workspace, workspace_bytes, cuda_stream);
}

int cgtp_message_field_bipartite(const float* node_feats, const int64_t* edge_index, const float* edge_feats,
                                 const float* W_edge, const float* W_node, const float* W_out, int lmax, int lmax_out, int N,
                                 int Ne, int C, const uint8_t* parity_mask, float* out, int64_t n_send, int64_t nodes,
                                 int64_t E, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    return field_entry(false, node_feats, edge_index, edge_feats, W_edge, W_node, W_out, lmax, lmax_out, N, Ne, C, parity_mask,
                       out, n_send, nodes, E, workspace, workspace_bytes, cuda_stream);
}

int cgtp_message_field_lw(const float* node_feats, const int64_t* edge_index, const float* edge_feats, const float* W_edge,
                          const float* W_node, const float* W_out, int lmax, int lmax_out, int N, int Ne, int C,
                          const uint8_t* parity_mask, float* out, int64_t nodes, int64_t E, void* workspace,
                          size_t workspace_bytes, void* cuda_stream)
{
    return field_entry(true, node_feats, edge_index, edge_feats, W_edge, W_node, W_out, lmax, lmax_out, N, Ne, C, parity_mask,
                       out, nodes, nodes, E, workspace, workspace_bytes, cuda_stream);
}

size_t cgtp_message_field_parity_workspace_bytes(int lmax, int lmax_out, int N, int Ne, int C, int64_t nodes, int64_t E)
{
    (void)N;
    (void)Ne;
    if (lmax < 0 || lmax_out < 0 || C <= 0 || nodes < 0 || E < 0) return 0;
    return field_ws_bytes(lmax, lmax_out, 4 * C, nodes, nodes, E);
}

int cgtp_message_field_parity(const float* node_feats, const int64_t* edge_index, const float* edge_feats,
                              const float* W_edge, const float* W_node, const float* W_out, int lmax, int lmax_out, int N,
                              int Ne, int C, float* out, int64_t nodes, int64_t E, void* workspace, size_t workspace_bytes,
                              void* cuda_stream)
{
    clear_error();
    if (C <= 0 || C > 256) { set_error("C=%d outside [1, 256] (4*C internal rank channels per pass)", C); return C <= 0 ? CGTP_ERR_INVALID : CGTP_ERR_UNSUPPORTED; }
    uint8_t mask[1024];
    for (int k = 0; k < 4 * C; ++k) mask[k] = k >= 2 * C;
    int rc = check_common(lmax, lmax_out, N, 4 * C, mask);
    if (rc) return rc;
    if (Ne <= 0) { set_error("Ne must be positive (Ne=%d)", Ne); return CGTP_ERR_INVALID; }
    if (nodes < 0 || E < 0) { set_error("negative size"); return CGTP_ERR_INVALID; }
    if (nodes == 0) return CGTP_OK;
    if (!node_feats || !W_edge || !W_node || !W_out || !out || !workspace || (E > 0 && (!edge_index || !edge_feats))) {
        set_error("null pointer argument");
        return CGTP_ERR_INVALID;
    }
    if (!aligned16(node_feats) || !aligned16(out) || !aligned16(W_edge) || !aligned16(W_node) || !aligned16(W_out) ||
        (E > 0 && (!aligned16(edge_index) || !aligned16(edge_feats))) || (reinterpret_cast<uintptr_t>(workspace) & 255u)) {
        set_error("misaligned pointer (tensors need 16-byte, workspace 256-byte alignment)");
        return CGTP_ERR_INVALID;
    }
    if (workspace_bytes < field_ws_bytes(lmax, lmax_out, 4 * C, nodes, nodes, E)) {
        set_error("workspace too small: %zu < %zu bytes", workspace_bytes, field_ws_bytes(lmax, lmax_out, 4 * C, nodes, nodes, E));
        return CGTP_ERR_INVALID;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const Plan* p = get_plan(lmax, lmax_out);
    if (!p) return CGTP_ERR_CUDA;
    const ParityPlan* pp = get_parity_plan(C, N, false);  // the run index 8 cat + 4 s1 + 2 s2 + tau of the on-site dispatch
    if (!pp) return CGTP_ERR_CUDA;
    const size_t nslot = (size_t)N * p->L2, eslot = (size_t)Ne * p->L2, sector = (size_t)N * p->Lo2;
    for (int ps = 0; ps < 4; ++ps) {
        const int s1 = ps >> 1, s2 = ps & 1;  // slot of the edge field (factor 1, R10) and of the node field (factor 2)
        FieldPass q;
        q.edge_feats = edge_feats + (size_t)s1 * eslot;
        q.x_bs_edge = (int64_t)2 * eslot;
        q.node_feats = node_feats + (size_t)s2 * nslot;
        q.x_bs_node = (int64_t)2 * nslot;
        q.W_edge = W_edge;
        q.W_node = W_node;
        q.idx_in = pp->idx_in(ps);
        q.W_out = W_out;
        q.ldw_out = C;
        q.idx_out_e = pp->idx_out(ps);
        q.idx_out_o = pp->idx_out(ps) + 2 * C;
        q.Ce = 2 * C;
        q.Co = 2 * C;
        q.out_e = out + (size_t)(s1 ^ s2) * sector;      // alpha: p = p1 p2 with l1+l2+l even -> slot s1 ^ s2 (Eq.(28) :236)
        q.out_o = out + (size_t)(1 ^ s1 ^ s2) * sector;  // beta: l1+l2+l odd -> the other slot
        q.o_bs = (int64_t)2 * sector;
        q.accumulate = ps > 0;
        q.sigma_C = C;
        q.segments_done = ps > 0;
        q.lw = false;
        rc = field_pass(p, N, Ne, q, edge_index, nodes, nodes, E, workspace, st);
        if (rc) return rc;
    }
    return CGTP_OK;
}

// ------------------------------------------------------------------------------ parity-slot entry points
size_t cgtp_onsite_parity_workspace_bytes(int lmax, int lmax_out, int N, int C, int64_t batch)
{
    (void)N;
    if (lmax < 0 || lmax_out < 0 || C <= 0 || batch < 0) return 0;
    return onsite_ws_bytes(lmax, lmax_out, 4 * C, batch);
}

int cgtp_onsite_parity(const float* A, const float* B, const float* W_a, const float* W_b, const float* W_out, int lmax,
                       int lmax_out, int N, int C, float* out, int64_t batch, void* workspace, size_t workspace_bytes,
                       void* cuda_stream)
{
    clear_error();
    if (C <= 0 || C > 256) { set_error("C=%d outside [1, 256] (4*C internal rank channels per pass)", C); return C <= 0 ? CGTP_ERR_INVALID : CGTP_ERR_UNSUPPORTED; }
    uint8_t mask[1024];
    for (int k = 0; k < 4 * C; ++k) mask[k] = k >= 2 * C;
    int rc = check_common(lmax, lmax_out, N, 4 * C, mask);
    if (rc) return rc;
    if (batch < 0) { set_error("negative batch"); return CGTP_ERR_INVALID; }
    if (batch == 0) return CGTP_OK;
    if (!A || !B || !W_a || !W_b || !W_out || !out || !workspace) { set_error("null pointer argument"); return CGTP_ERR_INVALID; }
    if (!aligned16(A) || !aligned16(B) || !aligned16(out) || !aligned16(W_a) || !aligned16(W_b) || !aligned16(W_out) ||
        (reinterpret_cast<uintptr_t>(workspace) & 255u)) {
        set_error("misaligned pointer (tensors need 16-byte, workspace 256-byte alignment)");
        return CGTP_ERR_INVALID;
    }
    if (workspace_bytes < onsite_ws_bytes(lmax, lmax_out, 4 * C, batch)) {
        set_error("workspace too small: %zu < %zu bytes", workspace_bytes, onsite_ws_bytes(lmax, lmax_out, 4 * C, batch));
        return CGTP_ERR_INVALID;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const Plan* p = get_plan(lmax, lmax_out);
    if (!p) return CGTP_ERR_CUDA;
    const ParityPlan* pp = get_parity_plan(C, N, false);
    if (!pp) return CGTP_ERR_CUDA;
    const size_t slot = (size_t)N * p->L2, sector = (size_t)N * p->Lo2;
    for (int ps = 0; ps < 4; ++ps) {
        const int s1 = ps >> 1, s2 = ps & 1;
        OnsitePass q;
        q.A = A + (size_t)s1 * slot;
        q.B = B + (size_t)s2 * slot;
        q.x_bs = (int64_t)2 * slot;
        q.W_a = W_a;
        q.W_b = W_b;
        q.idx_in = pp->idx_in(ps);
        q.W_out = W_out;
        q.ldw_out = C;
        q.idx_out_e = pp->idx_out(ps);
        q.idx_out_o = pp->idx_out(ps) + 2 * C;
        q.Ce = 2 * C;
        q.Co = 2 * C;
        q.out_e = out + (size_t)(s1 ^ s2) * sector;      // alpha: p = p1 p2 with l1+l2+l even -> slot s1 ^ s2
        q.out_o = out + (size_t)(1 ^ s1 ^ s2) * sector;  // beta: l1+l2+l odd -> the other slot
        q.o_bs = (int64_t)2 * sector;
        q.accumulate = ps > 0;  // pass (0,0) writes both sectors, the others add to them
        q.sigma_C = C;
        q.lw_in = q.lw_out = 0;
        rc = onsite_pass(p, N, q, batch, workspace, st);
        if (rc) return rc;
    }
    return CGTP_OK;
}

size_t cgtp_message_parity_workspace_bytes(int lmax, int lmax_out, int N, int C, int64_t nodes, int64_t E)
{
    (void)N;
    (void)E;
    if (lmax < 0 || lmax_out < 0 || C <= 0 || nodes < 0) return 0;
    return message_ws_bytes(lmax, lmax_out, 4 * C, 2 * C, nodes, nodes);
}

int cgtp_message_parity(const float* node_feats, const int64_t* edge_index, const float* edge_vec,
                        const float* edge_radial, const float* W_node, const float* W_out, int lmax, int lmax_out,
                        int N, int C, float* out, int64_t nodes, int64_t E, void* workspace, size_t workspace_bytes,
                        void* cuda_stream)
{
    clear_error();
    if (C <= 0 || C > 256) { set_error("C=%d outside [1, 256] (4*C internal rank channels per pass)", C); return C <= 0 ? CGTP_ERR_INVALID : CGTP_ERR_UNSUPPORTED; }
    uint8_t mask[1024];
    for (int k = 0; k < 4 * C; ++k) mask[k] = k >= 2 * C;
    int rc = check_common(lmax, lmax_out, N, 4 * C, mask);
    if (rc) return rc;
    rc = check_message_args(node_feats, edge_index, edge_vec, edge_radial, W_node, W_out, out, nodes, nodes, E, workspace);
    if (rc || nodes == 0) return rc;
    if (workspace_bytes < message_ws_bytes(lmax, lmax_out, 4 * C, 2 * C, nodes, nodes)) {
        set_error("workspace too small: %zu < %zu bytes", workspace_bytes, message_ws_bytes(lmax, lmax_out, 4 * C, 2 * C, nodes, nodes));
        return CGTP_ERR_INVALID;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const Plan* p = get_plan(lmax, lmax_out);
    if (!p) return CGTP_ERR_CUDA;
    const ParityPlan* pp = get_parity_plan(C, N, true);
    if (!pp) return CGTP_ERR_CUDA;
    const size_t slot = (size_t)N * p->L2, sector = (size_t)N * p->Lo2;
    for (int s_in = 0; s_in < 2; ++s_in) {
        MessagePass q;
        q.node_feats = node_feats + (size_t)s_in * slot;
        q.x_bs = (int64_t)2 * slot;
        q.W_node = W_node;
        q.idx_in = pp->idx_in(s_in);
        q.edge_radial = edge_radial;
        q.radial_stride = 8 * C;
        q.W_out = W_out;
        q.ldw_out = C;
        q.idx_out_e = pp->idx_out(s_in);
        q.idx_out_o = pp->idx_out(s_in) + 2 * C;
        q.Ce = 2 * C;
        q.Co = 2 * C;
        q.out_e = out + (size_t)s_in * sector;        // Eq.(45): alpha reads the slot of its output sector
        q.out_o = out + (size_t)(1 - s_in) * sector;  // Eq.(56): beta reads the opposite slot
        q.o_bs = (int64_t)2 * sector;
        q.accumulate = s_in > 0;
        q.sigma_C = C;
        q.segments_done = s_in > 0;
        q.lw_in = q.lw_out = 0;
        q.radial_l1 = false;
        rc = message_pass(p, N, q, edge_index, edge_vec, nodes, nodes, E, workspace, st);
        if (rc) return rc;
    }
    return CGTP_OK;
}

// ------------------------------------------------------------------------------ host-buffer entry points
// The host entry points allocate from the stream-ordered pool; without a release threshold the pool hands its
// memory back to the driver at every synchronisation and the next call pays for a fresh allocation.
static void keep_pool_memory()
{
    static bool done[64] = {false};
    const int dev = current_device();
    if (dev < 0 || dev >= 64 || done[dev]) return;
    cudaMemPool_t pool;
    if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
        uint64_t keep = UINT64_MAX;
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
    done[dev] = true;
}

// Streams, events and chunk buffers of cgtp_onsite_host live for the life of the process (grow-only): creating and
// destroying them per call cost more than a millisecond of the 3.4 ms end-to-end step.
namespace {
constexpr int kHostStreams = 4;
struct HostCtx {
    std::mutex mu;
    bool ready = false;
    // one stream per engine, so that a host->device copy never queues behind a device->host copy of an earlier chunk
    // (copies of one direction execute in issue order: with a stream per chunk the H2D engine stalled on them)
    cudaStream_t s_h2d, s_comp, s_d2h;
    cudaEvent_t start, ev_h2d[kHostStreams], ev_comp[kHostStreams], ev_d2h[kHostStreams], ev_end;
    float *dA[kHostStreams] = {}, *dB[kHostStreams] = {}, *dO[kHostStreams] = {};
    void* dws = nullptr;  // one workspace: the chunks' kernels run in order on s_comp
    size_t in_bytes = 0, out_bytes = 0, ws_bytes = 0;
    float* dW = nullptr;  // W_a | W_b | W_out
    size_t w_bytes = 0;
};
HostCtx g_host[64];  // one per CUDA device ordinal

int host_ctx_reserve(HostCtx& h, size_t in_bytes, size_t out_bytes, size_t ws_bytes, size_t w_bytes)
{
    if (!h.ready) {
        CGTP_CUDA_CHECK(cudaStreamCreateWithFlags(&h.s_h2d, cudaStreamNonBlocking));
        CGTP_CUDA_CHECK(cudaStreamCreateWithFlags(&h.s_comp, cudaStreamNonBlocking));
        CGTP_CUDA_CHECK(cudaStreamCreateWithFlags(&h.s_d2h, cudaStreamNonBlocking));
        for (int s = 0; s < kHostStreams; ++s) {
            CGTP_CUDA_CHECK(cudaEventCreateWithFlags(&h.ev_h2d[s], cudaEventDisableTiming));
            CGTP_CUDA_CHECK(cudaEventCreateWithFlags(&h.ev_comp[s], cudaEventDisableTiming));
            CGTP_CUDA_CHECK(cudaEventCreateWithFlags(&h.ev_d2h[s], cudaEventDisableTiming));
        }
        CGTP_CUDA_CHECK(cudaEventCreateWithFlags(&h.start, cudaEventDisableTiming));
        CGTP_CUDA_CHECK(cudaEventCreateWithFlags(&h.ev_end, cudaEventDisableTiming));
        h.ready = true;
    }
    if (in_bytes > h.in_bytes || out_bytes > h.out_bytes || ws_bytes > h.ws_bytes) {
        CGTP_CUDA_CHECK(cudaDeviceSynchronize());
        for (int s = 0; s < kHostStreams; ++s) {
            cudaFree(h.dA[s]); cudaFree(h.dB[s]); cudaFree(h.dO[s]);
            h.dA[s] = h.dB[s] = h.dO[s] = nullptr;
        }
        cudaFree(h.dws);
        h.dws = nullptr;
        h.in_bytes = std::max(h.in_bytes, in_bytes);
        h.out_bytes = std::max(h.out_bytes, out_bytes);
        h.ws_bytes = std::max(h.ws_bytes, ws_bytes);
        for (int s = 0; s < kHostStreams; ++s) {
            CGTP_CUDA_CHECK(cudaMalloc(&h.dA[s], h.in_bytes));
            CGTP_CUDA_CHECK(cudaMalloc(&h.dB[s], h.in_bytes));
            CGTP_CUDA_CHECK(cudaMalloc(&h.dO[s], h.out_bytes));
        }
        CGTP_CUDA_CHECK(cudaMalloc(&h.dws, h.ws_bytes));
    }
    if (w_bytes > h.w_bytes) {
        CGTP_CUDA_CHECK(cudaDeviceSynchronize());
        cudaFree(h.dW);
        h.dW = nullptr;
        CGTP_CUDA_CHECK(cudaMalloc(&h.dW, w_bytes));
        h.w_bytes = w_bytes;
    }
    return CGTP_OK;
}
}  // namespace

int cgtp_onsite_host(const float* A, const float* B, const float* W_a, const float* W_b, const float* W_out, int lmax,
                     int lmax_out, int N, int C, const uint8_t* parity_mask, float* out, int64_t batch,
                     void* cuda_stream)
{
    clear_error();
    int rc = check_common(lmax, lmax_out, N, C, parity_mask);
    if (rc) return rc;
    if (batch < 0) { set_error("negative batch"); return CGTP_ERR_INVALID; }
    if (batch == 0) return CGTP_OK;
    if (!A || !B || !W_a || !W_b || !W_out || !out) { set_error("null pointer argument"); return CGTP_ERR_INVALID; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const size_t L2 = (size_t)(lmax + 1) * (lmax + 1), Lo2 = (size_t)(lmax_out + 1) * (lmax_out + 1);
    const size_t wfl = (size_t)C * N;  // floats per weight matrix
    const size_t in_per = (size_t)N * L2 * 4, out_per = (size_t)2 * N * Lo2 * 4;
    // Batch chunks: in steady state the H2D copy of chunk k+1, the kernels of chunk k and the D2H copy of chunk k-1 run
    // together (PCIe is full duplex; 55 GB/s per direction alone, 48 GB/s each when both run, measured).  Every copy
    // has a fixed cost, so the chunks are few and large in the middle and small at both ends, where the first H2D and
    // the last D2H have nothing to overlap with: fractions 2 6 8 8 6 2 of 32 (2.83 ms at configs[1]; ten chunks
    // 1 1 2 4 8 8 4 2 1 1 took 2.95 ms, sixteen equal ones 3.1 ms).
    static const int kFrac[] = {2, 6, 8, 8, 6, 2};
    constexpr int kNumFrac = (int)(sizeof(kFrac) / sizeof(kFrac[0]));
    int64_t unit = (batch + 31) / 32;
    if (unit < 16) unit = 16;
    const int64_t chunk = std::min<int64_t>(batch, 8 * unit);  // largest chunk: sizes the buffers
    const size_t wsb = onsite_ws_bytes(lmax, lmax_out, C, chunk);

    const int dev = current_device();
    if (dev < 0 || dev >= 64) { set_error("no current CUDA device"); return CGTP_ERR_CUDA; }
    HostCtx& h = g_host[dev];
    std::lock_guard<std::mutex> lock(h.mu);
    rc = host_ctx_reserve(h, (size_t)chunk * in_per, (size_t)chunk * out_per, wsb, 3 * wfl * 4);
    if (rc) return rc;
    float *dWa = h.dW, *dWb = h.dW + wfl, *dWo = h.dW + 2 * wfl;
    CGTP_CUDA_CHECK(cudaMemcpyAsync(dWa, W_a, wfl * 4, cudaMemcpyHostToDevice, st));
    CGTP_CUDA_CHECK(cudaMemcpyAsync(dWb, W_b, wfl * 4, cudaMemcpyHostToDevice, st));
    CGTP_CUDA_CHECK(cudaMemcpyAsync(dWo, W_out, wfl * 4, cudaMemcpyHostToDevice, st));
    CGTP_CUDA_CHECK(cudaEventRecord(h.start, st));
    CGTP_CUDA_CHECK(cudaStreamWaitEvent(h.s_h2d, h.start, 0));
    CGTP_CUDA_CHECK(cudaStreamWaitEvent(h.s_comp, h.start, 0));
    int k = 0;
    for (int64_t b0 = 0, nb = 0; b0 < batch; b0 += nb, ++k) {
        const int s = k % kHostStreams;  // buffer set of this chunk
        nb = (k < kNumFrac ? kFrac[k] : 8) * unit;
        if (nb > batch - b0) nb = batch - b0;
        // inputs: the buffer set is free once the kernels of the chunk that used it last have run
        if (k >= kHostStreams) CGTP_CUDA_CHECK(cudaStreamWaitEvent(h.s_h2d, h.ev_comp[s], 0));
        CGTP_CUDA_CHECK(cudaMemcpyAsync(h.dA[s], A + (size_t)b0 * N * L2, nb * in_per, cudaMemcpyHostToDevice, h.s_h2d));
        CGTP_CUDA_CHECK(cudaMemcpyAsync(h.dB[s], B + (size_t)b0 * N * L2, nb * in_per, cudaMemcpyHostToDevice, h.s_h2d));
        CGTP_CUDA_CHECK(cudaEventRecord(h.ev_h2d[s], h.s_h2d));
        // kernels: need the inputs, and the output buffer back from the copy of the chunk that used it last
        CGTP_CUDA_CHECK(cudaStreamWaitEvent(h.s_comp, h.ev_h2d[s], 0));
        if (k >= kHostStreams) CGTP_CUDA_CHECK(cudaStreamWaitEvent(h.s_comp, h.ev_d2h[s], 0));
        rc = cgtp_onsite(h.dA[s], h.dB[s], dWa, dWb, dWo, lmax, lmax_out, N, C, parity_mask, h.dO[s], nb, h.dws, wsb,
                         h.s_comp);
        if (rc) return rc;
        CGTP_CUDA_CHECK(cudaEventRecord(h.ev_comp[s], h.s_comp));
        // result
        CGTP_CUDA_CHECK(cudaStreamWaitEvent(h.s_d2h, h.ev_comp[s], 0));
        CGTP_CUDA_CHECK(cudaMemcpyAsync(out + (size_t)b0 * 2 * N * Lo2, h.dO[s], nb * out_per, cudaMemcpyDeviceToHost, h.s_d2h));
        CGTP_CUDA_CHECK(cudaEventRecord(h.ev_d2h[s], h.s_d2h));
    }
    CGTP_CUDA_CHECK(cudaEventRecord(h.ev_end, h.s_d2h));
    CGTP_CUDA_CHECK(cudaStreamWaitEvent(st, h.ev_end, 0));
    CGTP_CUDA_CHECK(cudaStreamSynchronize(st));
    return CGTP_OK;
}

int cgtp_message_host(const float* node_feats, const int64_t* edge_index, const float* edge_vec,
                      const float* edge_radial, const float* W_node, const float* W_out, int lmax, int lmax_out, int N,
                      int C, const uint8_t* parity_mask, float* out, int64_t nodes, int64_t E, void* cuda_stream)
{
    clear_error();
    int rc = check_common(lmax, lmax_out, N, C, parity_mask);
    if (rc) return rc;
    if (nodes < 0 || E < 0) { set_error("negative size"); return CGTP_ERR_INVALID; }
    if (nodes == 0) return CGTP_OK;
    if (!node_feats || !W_node || !W_out || !out || (E > 0 && (!edge_index || !edge_vec || !edge_radial))) {
        set_error("null pointer argument");
        return CGTP_ERR_INVALID;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    keep_pool_memory();
    const size_t L2 = (size_t)(lmax + 1) * (lmax + 1), Lo2 = (size_t)(lmax_out + 1) * (lmax_out + 1);
    const size_t xb = (size_t)nodes * N * L2 * 4, ob = (size_t)nodes * 2 * N * Lo2 * 4, wb = (size_t)C * N * 4;
    const size_t eib = (size_t)2 * (E > 0 ? E : 1) * 8, evb = (size_t)(E > 0 ? E : 1) * 3 * 4, erb = (size_t)(E > 0 ? E : 1) * C * 4;
    const size_t wsb = cgtp_message_workspace_bytes(lmax, lmax_out, N, C, parity_mask, nodes, E);
    // stream-ordered allocations, released on every exit path
    struct Pool {
        cudaStream_t st;
        std::vector<void*> ptrs;
        ~Pool()
        {
            for (void* q : ptrs) cudaFreeAsync(q, st);
        }
        int take(void** q, size_t bytes)
        {
            CGTP_CUDA_CHECK(cudaMallocAsync(q, bytes, st));
            ptrs.push_back(*q);
            return CGTP_OK;
        }
    } pool{st, {}};
    float *dX, *dO, *dWn, *dWo, *dEv, *dEr;
    int64_t* dEi;
    void* dws;
    if ((rc = pool.take((void**)&dX, xb)) || (rc = pool.take((void**)&dO, ob)) || (rc = pool.take((void**)&dWn, wb)) ||
        (rc = pool.take((void**)&dWo, wb)) || (rc = pool.take((void**)&dEi, eib)) || (rc = pool.take((void**)&dEv, evb)) ||
        (rc = pool.take((void**)&dEr, erb)) || (rc = pool.take(&dws, wsb)))
        return rc;
    CGTP_CUDA_CHECK(cudaMemcpyAsync(dX, node_feats, xb, cudaMemcpyHostToDevice, st));
    CGTP_CUDA_CHECK(cudaMemcpyAsync(dWn, W_node, wb, cudaMemcpyHostToDevice, st));
    CGTP_CUDA_CHECK(cudaMemcpyAsync(dWo, W_out, wb, cudaMemcpyHostToDevice, st));
    if (E > 0) {
        CGTP_CUDA_CHECK(cudaMemcpyAsync(dEi, edge_index, (size_t)2 * E * 8, cudaMemcpyHostToDevice, st));
        CGTP_CUDA_CHECK(cudaMemcpyAsync(dEv, edge_vec, (size_t)E * 3 * 4, cudaMemcpyHostToDevice, st));
        CGTP_CUDA_CHECK(cudaMemcpyAsync(dEr, edge_radial, (size_t)E * C * 4, cudaMemcpyHostToDevice, st));
    }
    rc = cgtp_message(dX, dEi, dEv, dEr, dWn, dWo, lmax, lmax_out, N, C, parity_mask, dO, nodes, E, dws, wsb, st);
    if (rc) return rc;
    CGTP_CUDA_CHECK(cudaMemcpyAsync(out, dO, ob, cudaMemcpyDeviceToHost, st));
    const int grc = cgtp_message_status(dws, st);  // synchronises the stream
    return grc;
}

// ------------------------------------------------------------------------------------------ math mode
int cgtp_set_math_mode(int mode)
{
    clear_error();
    if (mode < CGTP_MATH_FP32 || mode > CGTP_MATH_TF32) { set_error("unknown math mode %d", mode); return CGTP_ERR_INVALID; }
    cgtp::set_math_mode(mode);
    return CGTP_OK;
}
int cgtp_get_math_mode(void) { return cgtp::get_math_mode(); }

// ------------------------------------------------------------------------------------------ kernel path
int cgtp_set_kernel_path(int flags)
{
    clear_error();
    if (flags < 0 || flags > 511) { set_error("unknown kernel-path flags %d", flags); return CGTP_ERR_INVALID; }
    cgtp::set_kernel_path(flags);
    return CGTP_OK;
}
int cgtp_get_kernel_path(void) { return cgtp::kernel_path(); }

// ------------------------------------------------------------------------------------ instrumentation
int64_t cgtp_launch_count(void) { return cgtp::launch_count(); }
int cgtp_profile_kinds(void) { return K_COUNT; }
const char* cgtp_profile_kind_name(int kind) { return (kind >= 0 && kind < K_COUNT) ? kKindNames[kind] : ""; }
int cgtp_profile_enable(int on)
{
    cgtp::profile_enable(on != 0);
    return CGTP_OK;
}
int cgtp_profile_collect(double* ms, int64_t* launches) { return cgtp::profile_collect(ms, launches); }

}  // extern "C"
