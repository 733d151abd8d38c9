/*
 * cgtp.h -- C ABI of libcgtp: B200-native (sm_100a) contracted Clebsch-Gordan tensor products.
 *
 * The hot path of the SCALE-CG method (arxiv 2605.15073; citations "PAPER.md:<line>" refer to the
 * paper text): the O(L^3) contracted Clebsch-Gordan tensor product at fixed CP rank, evaluated on a
 * Gauss-Legendre (theta) x Fourier (phi) grid.
 *
 * Conventions ("Readings"):
 *   - real spherical harmonics of Eq.(C1), orthonormal on S^2, no Condon-Shortley
 *     phase, coefficient order m = -l..l, flat index l*l + l + m;
 *   - all tensors row-major contiguous FP32; "device" pointers are CUDA device memory owned by the
 *     caller (e.g. allocated by PyTorch), 16-byte aligned; the library never frees caller memory;
 *   - parity_mask is a HOST array of C bytes: 0 = parity-even rank channel (pointwise grid product,
 *     Gaunt coupling, Eq.(38) :332), 1 = parity-odd rank channel (surface-curl pairing
 *     r.[grad A x grad B], Eq.(11)-(12) :107-:111, Eq.(57) :443).  It is structural (it selects the
 *     kernels that run), like lmax;
 *   - out has two parity sectors: sector 0 = sum over even channels (natural parity (-1)^l),
 *     sector 1 = sum over odd channels (opposite parity); out is fully overwritten;
 *   - every call is asynchronous on `cuda_stream` (a cudaStream_t passed as void*; NULL = legacy
 *     default stream) and does no host synchronisation, except where stated;
 *   - results are bitwise reproducible run to run (no floating-point atomics anywhere).
 *
 * Return codes: CGTP_OK, or
 *   CGTP_ERR_INVALID      null pointer, negative size, lmax < 0, lmax_out > 2*lmax, mask entry not in
 *                         {0,1}, misaligned pointer, workspace too small;
 *   CGTP_ERR_UNSUPPORTED  band limit above cgtp_max_lmax(), N or C above the compiled limits;
 *   CGTP_ERR_CUDA         a CUDA runtime call failed (message in cgtp_last_error());
 *   CGTP_ERR_GRAPH        edge_index not receiver-sorted or out of range (reported by
 *                         cgtp_message_status / cgtp_build_segments' status word).
 * No exception or abort ever crosses this boundary.
 */
#ifndef CGTP_H
#define CGTP_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CGTP_OK 0
#define CGTP_ERR_INVALID 1
#define CGTP_ERR_UNSUPPORTED 2
#define CGTP_ERR_CUDA 3
#define CGTP_ERR_GRAPH 4

/* Library version (major*10000 + minor*100 + patch). */
int cgtp_version(void);

/* Message of the last error raised on the calling thread ("" if none). Never NULL. */
const char* cgtp_last_error(void);

/* Largest band limit max(lmax, lmax_out) the compiled kernels support. */
int cgtp_max_lmax(void);

/* Quadrature grid used for (lmax, lmax_out): U Gauss-Legendre nodes in cos(theta) and V uniform
 * azimuths, U = ceil((2 lmax + lmax_out + 1)/2), V = 2 lmax + lmax_out + 1 -- the exactness bound of
 * PAPER.md:173 (U >= (3 lmax+1)/2, V >= 3 lmax+1) generalised to lmax_out != lmax. */
int cgtp_grid_shape(int lmax, int lmax_out, int* U, int* V);

/* ---------------------------------------------------------------------------------------------
 * On-site bilinear contraction, Eq.(1) at CP rank C, Eq.(3) (:39), natural-parity
 * inputs; the structured-grid pipeline of Sec. VII B, Eq.(35)-(41) (:322-:346), with the surface-curl
 * pairing Eq.(12) (:111) for the odd channels (Sec. VII C e, :469):
 *
 *   Ha[b,c,:] = W_a[c,:] . A[b]     Hb[b,c,:] = W_b[c,:] . B[b]                       (Eq.(35))
 *   even c:  T[b,c,lm] = int (Ha~ Hb~) Y_lm dOmega                                     (Eq.(36)-(40))
 *   odd  c:  T[b,c,lm] = int r.[grad Ha~ x grad Hb~] Y_lm dOmega   (A factor 1, B factor 2)
 *   out[b,s,n,lm] = sum_{c: mask[c]=s} W_out[n,c] T[b,c,lm],   l <= lmax_out           (Eq.(41))
 *
 * A, B      device [batch, N, (lmax+1)^2]
 * W_a, W_b  device [C, N]        W_out  device [N, C]
 * parity_mask  HOST [C]
 * out       device [batch, 2, N, (lmax_out+1)^2]
 * workspace device, >= cgtp_onsite_workspace_bytes(...) bytes, 256-byte aligned; contents are
 *           scratch (projected coefficients H and rank-space results T) and may be reused by the
 *           next call on the same stream.
 * batch may be 0 (no work, CGTP_OK).  0 <= lmax_out <= 2*lmax.
 * ------------------------------------------------------------------------------------------- */
size_t cgtp_onsite_workspace_bytes(int lmax, int lmax_out, int N, int C, int64_t batch);

int cgtp_onsite(const float* A, const float* B, const float* W_a, const float* W_b, const float* W_out,
                int lmax, int lmax_out, int N, int C, const uint8_t* parity_mask, float* out,
                int64_t batch, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * cgtp_onsite for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc).  Same operation, arguments, layouts and sectors as cgtp_onsite (Eq.(35)-(41)
 * PAPER.md:322-346, odd channels Eq.(11)-(12) :107-:111), but NO workspace argument and NO allocation of any kind: the
 * projected coefficients H and the rank-space results T live in a file-scope device array of
 * CGTP_STATIC_SCRATCH_BYTES (16 MiB; every GPU that loads the library's module holds it until the process exits), the
 * tables travel as kernel parameters, and the call makes no cudaMalloc / cudaFree / allocating library call and touches
 * no plan cache of the library (first call included).
 *
 * Limits: max(lmax, lmax_out) <= 4 and C <= 256 (any N, any batch: persistent CTAs walk the batch); beyond them
 * CGTP_ERR_UNSUPPORTED with a message naming the limit -- use cgtp_onsite with a workspace there.  Other errors as
 * cgtp_onsite.  One plain FP32 kernel (no TMA, no tensor cores, math mode ignored): made for small shapes, not for speed.
 *
 * ALL CALLS SHARE THE ONE ARRAY.  It keeps the last call's contents; no call reads a word it has not written itself, so
 * nothing needs clearing.  Calls that overlap on the GPU (different streams, concurrently replayed graphs) RACE on it;
 * calls on one stream are ordered and safe.  Asynchronous on cuda_stream.  Not counted by cgtp_launch_count / profiling.
 * ------------------------------------------------------------------------------------------- */
#define CGTP_STATIC_SCRATCH_BYTES (16u << 20)
int cgtp_onsite_static(const float* A, const float* B, const float* W_a, const float* W_b, const float* W_out,
                       int lmax, int lmax_out, int N, int C, const uint8_t* parity_mask, float* out,
                       int64_t batch, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Two feature fields (Eq.(28) :236, Sec. VI E :232-:240, Sec. VII C f :471):
 * "the deeper message-passing variant in which the edge-side message ... no longer factors as R.Y", written with
 * an edge field I^(E)[e, n1, l1 m1] and a node field I^(N)[j, n2, l2 m2].  At fixed CP rank (Eq.(3) :39; "an
 * explicit radial contraction is required on the edge side, replacing R~ by an analogue of Eq.(47)", :471):
 *
 *   a[e,c,:]      = W_edge[c,:] . edge_feats[e]                                  (factor 1)
 *   H[j,c,:]      = W_node[c,:] . node_feats[j]                                  (factor 2, Eq.(47) :398)
 *   T[i,c,lm]     = sum_{e: recv(e)=i} int P(a~[e,c], H~[send(e),c])(Omega) Y_lm dOmega
 *                   P = pointwise product (parity_mask[c] = 0, Category alpha, Eq.(52) :415) or the surface-curl
 *                   pairing {a~, H~} (parity_mask[c] = 1, Category beta, Eq.(57) :443; the edge field is factor 1)
 *   out[i,s,n,lm] = sum_{c: mask[c]=s} W_out[n,c] T[i,c,lm]                      (Eq.(55), (58))
 *
 * Both fields sit in their natural-parity slots and the weights are l-shared; sector 0 / 1 of `out` as in
 * cgtp_message.  Every edge is one fused synthesis-product-analysis pass (the grids stay on chip); the per-edge
 * coefficients are pooled per receiver in edge order (fixed order, no float atomics, bitwise reproducible).
 *
 * node_feats device [nodes, N, (lmax+1)^2]      edge_feats device [E, Ne, (lmax+1)^2]
 * edge_index device int64 [2, E], row 0 sender, row 1 receiver, receiver-sorted (validated on the device: query
 *            cgtp_message_status(workspace, stream); on CGTP_ERR_GRAPH `out` is undefined)
 * W_edge device [C, Ne]    W_node device [C, N]    W_out device [N, C]    parity_mask HOST [C]
 * out    device [nodes, 2, N, (lmax_out+1)^2]; receivers without in-edges get zeros
 * workspace device, >= cgtp_message_field_workspace_bytes(...) bytes, 256-byte aligned (scratch; edges are
 *           processed in chunks of at most 2^22 / C, so the size is bounded in E)
 * nodes or E may be 0.  Errors as cgtp_message.  Asynchronous on cuda_stream.
 * ------------------------------------------------------------------------------------------- */
size_t cgtp_message_field_workspace_bytes(int lmax, int lmax_out, int N, int Ne, int C, int64_t nodes, int64_t E);

int cgtp_message_field(const float* node_feats, const int64_t* edge_index, const float* edge_feats, const float* W_edge,
                       const float* W_node, const float* W_out, int lmax, int lmax_out, int N, int Ne, int C,
                       const uint8_t* parity_mask, float* out, int64_t nodes, int64_t E, void* workspace,
                       size_t workspace_bytes, void* cuda_stream);

/* The same coupling in the paper's own parameterisation, l-dependent CP weights (c_{cnl} of Eq.(35) :322 / Eq.(47) :398 on
 * both fields, lambda_c^{(nl)} of Eq.(41) :346 / Eq.(55) :427 on the output), as cgtp_message_lw:
 * W_edge device [lmax+1, C, Ne], W_node device [lmax+1, C, N], W_out device [lmax_out+1, N, C]; the matrix of degree l
 * acts on the coefficients l^2 .. l^2 + 2l.  Workspace: cgtp_message_field_workspace_bytes.  Everything else as
 * cgtp_message_field. */
int cgtp_message_field_lw(const float* node_feats, const int64_t* edge_index, const float* edge_feats, const float* W_edge,
                          const float* W_node, const float* W_out, int lmax, int lmax_out, int N, int Ne, int C,
                          const uint8_t* parity_mask, float* out, int64_t nodes, int64_t E, void* workspace,
                          size_t workspace_bytes, void* cuda_stream);

/* Bipartite form (one shard of a receiver-partitioned graph, as cgtp_message_bipartite): senders index node_feats
 * [n_send, N, (lmax+1)^2] (all nodes, after the all-gather), receivers are the local rows 0 .. nodes-1 of
 * out [nodes, 2, N, (lmax_out+1)^2]; edge_index row 0 in [0, n_send), row 1 in [0, nodes), receiver-sorted;
 * edge_feats [E, Ne, (lmax+1)^2] holds the shard's in-edges.  cgtp_message_field is the case n_send = nodes, and the
 * shards' outputs are the rows of the single call bit for bit (the per-receiver arithmetic does not depend on the
 * shard as long as no receiver's edges are split between edge chunks differently, i.e. E <= 2^22 / C per shard
 * and in the single call; otherwise equal within rounding). */
size_t cgtp_message_field_bipartite_workspace_bytes(int lmax, int lmax_out, int N, int Ne, int C, int64_t n_send,
                                                    int64_t nodes, int64_t E);

int cgtp_message_field_bipartite(const float* node_feats, const int64_t* edge_index, const float* edge_feats,
                                 const float* W_edge, const float* W_node, const float* W_out, int lmax, int lmax_out, int N,
                                 int Ne, int C, const uint8_t* parity_mask, float* out, int64_t n_send, int64_t nodes,
                                 int64_t E, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * nu-body on-site product (end of Sec. VI): "The grid pointwise product
 * extends to nu-body features through additional pointwise multiplications on the grid followed by a single
 * inverse transform", on the grid U = ceil((nu lmax + lmax_out + 1)/2), V = nu lmax + lmax_out + 1 that the
 * degree-(nu lmax + lmax_out) integrand needs ("tighten this requirement linearly in the body order nu"):
 *
 *   H(s)[b,c,:] = W_in[s][c,:] . X[s][b]                     s = 1..nu                  (Eq.(35) per factor)
 *   T[b,c,lm]   = int prod_s H(s)~[b,c](Omega) Y_lm dOmega   l <= lmax_out              (Eq.(36)-(40))
 *   out[b,n,lm] = sum_c W_out[n,c] T[b,c,lm]                                            (Eq.(41))
 *
 * Pointwise (parity-even) rank channels only -- the curl pairing is bilinear and the paper gives no nu-body
 * form of it -- so there is one output sector (natural parity).  nu = 2 equals sector 0 of cgtp_onsite with an
 * all-even mask.
 *
 * X      device [nu, batch, N, (lmax+1)^2]     W_in  device [nu, C, N]     W_out  device [N, C]
 * out    device [batch, N, (lmax_out+1)^2]
 * workspace device, >= cgtp_onsite_nbody_workspace_bytes(...) bytes, 256-byte aligned (scratch)
 * 1 <= nu <= 4, max(lmax, lmax_out) <= cgtp_max_lmax() (CGTP_ERR_UNSUPPORTED beyond, and where fewer than four columns of
 * the nu fields fit the shared memory of an SM: nu = 4 at band limit 20), 0 <= lmax_out <= nu*lmax
 * (CGTP_ERR_INVALID otherwise).  batch may be 0.  Asynchronous on cuda_stream, bitwise reproducible.
 * ------------------------------------------------------------------------------------------- */
size_t cgtp_onsite_nbody_workspace_bytes(int nu, int lmax, int lmax_out, int N, int C, int64_t batch);

int cgtp_onsite_nbody(const float* X, const float* W_in, const float* W_out, int nu, int lmax, int lmax_out,
                      int N, int C, float* out, int64_t batch, void* workspace, size_t workspace_bytes,
                      void* cuda_stream);

/* Grid of the nu-body product (cgtp_grid_shape is the case nu = 2). */
int cgtp_grid_shape_nu(int lmax, int lmax_out, int nu, int* U, int* V);

/* ---------------------------------------------------------------------------------------------
 * Parity-aware message passing, Eq.(2), pipeline of Sec. VII C, Eq.(46)-(59)
 * (:396-:453), natural-parity node features (Cases A and B, :197-:217), l1-shared radial factor:
 *
 *   H[j,c,:]  = W_node[c,:] . node_feats[j]                                            (Eq.(47))
 *   edge field (factor 1)  E_e(Omega) = edge_radial[e,c] * sum_{l1<=lmax,m1} Y_{l1m1}(r_e) Y_{l1m1}(Omega)
 *                                                                                     (Eq.(46),(48),(50))
 *   even c:  S[i,c,Omega] = sum_{e: recv(e)=i} E_e(Omega) H~[send(e),c](Omega)            (Eq.(52))
 *   odd  c:  S[i,c,Omega] = sum_e r.[grad E_e x grad H~[send(e),c]](Omega)                (Eq.(57))
 *   T[i,c,lm] = int S[i,c] Y_lm dOmega  (once per receiver, Eq.(53)-(54))
 *   out[i,s,n,lm] = sum_{c: mask[c]=s} W_out[n,c] T[i,c,lm]                            (Eq.(55),(58),(59))
 *
 * node_feats  device [nodes, N, (lmax+1)^2]
 * edge_index  device int64 [2, E]: row 0 = sender j, row 1 = receiver i; sorted by receiver
 *             (ascending, ties in any fixed order -- the order of the sum within a receiver is the
 *             input order, which makes the result bitwise reproducible)
 * edge_vec    device [E, 3] = r_j - r_i; only the direction is used; must be non-zero
 * edge_radial device [E, C] = R~ of Eq.(46), computed by the caller
 * W_node      device [C, N]      W_out  device [N, C]      parity_mask  HOST [C]
 * out         device [nodes, 2, N, (lmax_out+1)^2]; receivers without edges get zeros
 * workspace   device, >= cgtp_message_workspace_bytes(...) bytes, 256-byte aligned
 *
 * Graph errors are detected on the device: the call still returns CGTP_OK, out is zero-filled, and
 * cgtp_message_status() returns CGTP_ERR_GRAPH.
 * ------------------------------------------------------------------------------------------- */
size_t cgtp_message_workspace_bytes(int lmax, int lmax_out, int N, int C, const uint8_t* parity_mask,
                                    int64_t nodes, int64_t E);

int cgtp_message(const float* node_feats, const int64_t* edge_index, const float* edge_vec,
                 const float* edge_radial, const float* W_node, const float* W_out,
                 int lmax, int lmax_out, int N, int C, const uint8_t* parity_mask, float* out,
                 int64_t nodes, int64_t E, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Bipartite form of cgtp_message, the building block of receiver sharding: the
 * sum of Eq.(2) runs over the in-edges of the n_recv receivers this call owns, while the
 * senders j index a (possibly larger) set of n_send nodes whose features are given.
 *   node_feats  device [n_send, N, (lmax+1)^2]
 *   edge_index  device int64 [2, E]: row 0 = sender in [0, n_send), row 1 = receiver in [0, n_recv),
 *               sorted by receiver
 *   out         device [n_recv, 2, N, (lmax_out+1)^2]
 * Everything else as cgtp_message, which is the case n_send = n_recv = nodes. */
size_t cgtp_message_bipartite_workspace_bytes(int lmax, int lmax_out, int N, int C, const uint8_t* parity_mask,
                                              int64_t n_send, int64_t n_recv, int64_t E);

int cgtp_message_bipartite(const float* node_feats, const int64_t* edge_index, const float* edge_vec,
                           const float* edge_radial, const float* W_node, const float* W_out,
                           int lmax, int lmax_out, int N, int C, const uint8_t* parity_mask, float* out,
                           int64_t n_send, int64_t n_recv, int64_t E, void* workspace, size_t workspace_bytes,
                           void* cuda_stream);

/* Synchronises `cuda_stream` and returns the graph status the last cgtp_message on this workspace
 * left: CGTP_OK or CGTP_ERR_GRAPH (CGTP_ERR_CUDA if the stream reports an error). */
int cgtp_message_status(const void* workspace, void* cuda_stream);

/* Segmentation step of cgtp_message on its own (integer work, bit-exact):
 * row_ptr[i] = index of the first edge whose receiver is >= i, row_ptr[nodes] = E.
 * edge_index device int64 [2,E]; row_ptr device int64 [nodes+1]; status device int32 [1], set to
 * CGTP_OK or CGTP_ERR_GRAPH (receivers not ascending, or a sender/receiver outside [0,nodes)). */
int cgtp_build_segments(const int64_t* edge_index, int64_t E, int64_t nodes, int64_t* row_ptr,
                        int32_t* status, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Parity-labelled inputs (Sec. VI :193-:240; pipelines Sec. VII C a-c :383-:453 and e :469).
 *
 * Features carry a parity label p = +-1 next to l (Eq.(2) :33: I_{j n2 l2 m2, p2}).  Storage: a slot axis of
 * length 2 in front of the channel axis, slot 0 = the natural-parity part p = (-1)^l, slot 1 = the
 * opposite-parity part p = -(-1)^l (the paper's +1 / -1 slots, indexed relative to (-1)^l); `out` has the same
 * two slots (they are the two sectors of cgtp_onsite / cgtp_message).  The output parity is p = p1 p2 (:29).
 * Every output sector (l, p) is the sum of a Category-alpha run (direct Gaunt coupling, l1+l2+l even, Cases A
 * and C) and a Category-beta run (surface curl, l1+l2+l odd, Cases B and D), Eq.(59); by the slot rules
 * Eq.(44)-(45) an alpha run reads the source slot of its output sector and by Eq.(56) a beta run the other one.
 * Each run has its own CP weights (Eq.(42)-(43), "fitted independently" :381, :437) and feeds only the output
 * degrees with (-1)^l = sigma (Eq.(54)-(55)); tau = 0 for sigma = +1 (even l), 1 for sigma = -1 (odd l);
 * cat = 0 alpha, 1 beta.
 *
 * cgtp_message_parity: run r = 4*cat + 2*s_out + tau (8 runs; the paper's (p, sigma) is (s_out, tau) with
 * p = (-1)^{s_out} sigma); cost 4 alpha + 4 beta runs = the 12x of Eq.(60).
 *   node_feats  device [nodes, 2, N, (lmax+1)^2]
 *   edge_radial device [E, 8, C]  = R~ of Eq.(46) for every run
 *   W_node      device [8, C, N]      W_out  device [8, N, C]
 *   out         device [nodes, 2, N, (lmax_out+1)^2], fully overwritten
 *   edge_index, edge_vec, workspace, graph status: as cgtp_message.  4*C <= 1024.
 * cgtp_onsite_parity (VII C e): run r = 8*cat + 4*s1 + 2*s2 + tau over the slots s1 of A and s2 of B (16 runs,
 * the paper's 24x); the run's alpha part lands in sector s1^s2, its beta part in sector 1^s1^s2.
 *   A, B        device [batch, 2, N, (lmax+1)^2]
 *   W_a, W_b    device [16, C, N]     W_out  device [16, N, C]
 *   out         device [batch, 2, N, (lmax_out+1)^2], fully overwritten
 * ------------------------------------------------------------------------------------------- */
size_t cgtp_onsite_parity_workspace_bytes(int lmax, int lmax_out, int N, int C, int64_t batch);

int cgtp_onsite_parity(const float* A, const float* B, const float* W_a, const float* W_b, const float* W_out,
                       int lmax, int lmax_out, int N, int C, float* out, int64_t batch, void* workspace,
                       size_t workspace_bytes, void* cuda_stream);

size_t cgtp_message_parity_workspace_bytes(int lmax, int lmax_out, int N, int C, int64_t nodes, int64_t E);

int cgtp_message_parity(const float* node_feats, const int64_t* edge_index, const float* edge_vec,
                        const float* edge_radial, const float* W_node, const float* W_out,
                        int lmax, int lmax_out, int N, int C, float* out, int64_t nodes, int64_t E,
                        void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * l-dependent CP weights, the paper's own parameterisation (c_{cnl} in Eq.(35) PAPER.md:322 and Eq.(47) :398,
 * lambda_c^{(nl)} in Eq.(41) :346 and Eq.(55) :427; cgtp_onsite / cgtp_message take one matrix for all degrees):
 *   H[b,c,lm] = sum_n W[l][c,n] A[b,n,lm]         out[b,s,n,lm] = sum_{c: mask[c]=s} W_out[l][n,c] T[b,c,lm]
 *   W_a, W_b, W_node  device [lmax+1, C, N]        W_out  device [lmax_out+1, N, C]
 * The radial factor of the edge stays l1-shared, edge_radial [E, C].  Every other argument, the workspace size
 * (cgtp_onsite_workspace_bytes / cgtp_message_workspace_bytes) and the error behaviour are those of cgtp_onsite /
 * cgtp_message.  The channel projections run once per degree l over the coefficient columns l^2 .. l^2 + 2l.
 * ------------------------------------------------------------------------------------------- */
int cgtp_onsite_lw(const float* A, const float* B, const float* W_a, const float* W_b, const float* W_out,
                   int lmax, int lmax_out, int N, int C, const uint8_t* parity_mask, float* out,
                   int64_t batch, void* workspace, size_t workspace_bytes, void* cuda_stream);

int cgtp_message_lw(const float* node_feats, const int64_t* edge_index, const float* edge_vec,
                    const float* edge_radial, const float* W_node, const float* W_out,
                    int lmax, int lmax_out, int N, int C, const uint8_t* parity_mask, float* out,
                    int64_t nodes, int64_t E, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Message passing in the paper's full parameterisation: the l-dependent weights of cgtp_message_lw AND the l1-dependent
 * radial factor R~_{jicl1} of Eq.(46): the edge field of channel c is
 *   E_{e,c}(Omega) = sum_{l1 <= lmax} edge_radial[e,c,l1] sum_{m1} Y_{l1m1}(r_e) Y_{l1m1}(Omega)          (Eq.(48), (50))
 * edge_radial  device [E, C, lmax+1]; everything else as cgtp_message_lw (same workspace size). */
int cgtp_message_lwr(const float* node_feats, const int64_t* edge_index, const float* edge_vec,
                     const float* edge_radial, const float* W_node, const float* W_out,
                     int lmax, int lmax_out, int N, int C, const uint8_t* parity_mask, float* out,
                     int64_t nodes, int64_t E, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Host-buffer entry points (end-to-end path): same semantics as cgtp_onsite / cgtp_message, but
 * every tensor pointer is HOST memory (pinned memory recommended; pageable works, slower).  The
 * library allocates device memory from the CUDA stream-ordered pool, copies inputs host->device in
 * batch chunks overlapped with compute, runs the device path, copies `out` device->host, and
 * synchronises before returning.  Returns CGTP_ERR_GRAPH directly for a bad graph.
 * ------------------------------------------------------------------------------------------- */
int cgtp_onsite_host(const float* A, const float* B, const float* W_a, const float* W_b, const float* W_out,
                     int lmax, int lmax_out, int N, int C, const uint8_t* parity_mask, float* out,
                     int64_t batch, void* cuda_stream);

int cgtp_message_host(const float* node_feats, const int64_t* edge_index, const float* edge_vec,
                      const float* edge_radial, const float* W_node, const float* W_out,
                      int lmax, int lmax_out, int N, int C, const uint8_t* parity_mask, float* out,
                      int64_t nodes, int64_t E, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Arithmetic of the channel projections (Eq.(35), Eq.(41) :346, Eq.(47) :398, Eq.(55) :427),
 * the dense GEMM-shaped stages of the path.  Process-wide, read at every call:
 *   CGTP_MATH_FP32    FP32 fused multiply-adds on the CUDA cores (default; the path the 1e-5 parity bar is
 *                     stated for);
 *   CGTP_MATH_3XTF32  tcgen05 tensor cores, every FP32 operand split into two TF32 terms, three MMAs per
 *                     product, FP32 accumulation in tensor memory (error ~1e-6 relative, reported separately);
 *   CGTP_MATH_TF32    tcgen05 tensor cores, single TF32 pass (error ~1e-3 relative; fails the parity bar by
 *                     design, for throughput comparison only).
 * Every other stage always runs in FP32.  cgtp_set_math_mode returns CGTP_ERR_INVALID for an unknown mode.
 * ------------------------------------------------------------------------------------------- */
#define CGTP_MATH_FP32 0
#define CGTP_MATH_3XTF32 1
#define CGTP_MATH_TF32 2
int cgtp_set_math_mode(int mode);
int cgtp_get_math_mode(void);

/* ---------------------------------------------------------------------------------------------
 * Two parity-bearing fields, Eq.(28) with the parity labels of both fields (Sec. VI E :232-:240,
 * Sec. VII C f :471: "The dispatch reads from both I^(E) and I^(N) with independent parity-slot selections at (l1,p1) and
 * (l2,p2) ... four input-parity combinations, two output-l parities, and Categories alpha and beta").  Slot axes as in
 * cgtp_onsite_parity (R19): slot 0 = natural parity (-1)^l, slot 1 = opposite parity.
 *
 *   run r = 8 cat + 4 s1 + 2 s2 + tau   (cat: 0 alpha = Gaunt coupling, 1 beta = surface-curl coupling; s1 / s2: slot of
 *                                        the edge field / the node field; tau: output-degree parity (-1)^l = sigma, Eq.(54))
 *   a_r[e,c,:] = W_edge[r,c,:] . edge_feats[e,s1]        H_r[j,c,:] = W_node[r,c,:] . node_feats[j,s2]
 *   T_r[i,c,lm] = sum_{e -> i} coupling_cat(a_r[e,c], H_r[send(e),c])_lm   kept at the degrees l with (l & 1) == tau
 *   out[i, s, n, lm] += sum_c W_out[r,n,c] T_r[i,c,lm]   with s = s1 ^ s2 (alpha) or 1 ^ s1 ^ s2 (beta): p = p1 p2 (:236)
 *
 * node_feats device [nodes, 2, N, (lmax+1)^2]     edge_feats device [E, 2, Ne, (lmax+1)^2]
 * W_edge device [16, C, Ne]   W_node device [16, C, N]   W_out device [16, N, C]
 * out device [nodes, 2, N, (lmax_out+1)^2], fully overwritten; everything else as cgtp_message_field.  Four passes of the
 * two-field pipeline over 4 C internal rank channels (cost: the paper's upper bound 24 x, Eq.(61)); C <= 256.
 * ------------------------------------------------------------------------------------------- */
size_t cgtp_message_field_parity_workspace_bytes(int lmax, int lmax_out, int N, int Ne, int C, int64_t nodes, int64_t E);
int cgtp_message_field_parity(const float* node_feats, const int64_t* edge_index, const float* edge_feats,
                              const float* W_edge, const float* W_node, const float* W_out,
                              int lmax, int lmax_out, int N, int Ne, int C, float* out,
                              int64_t nodes, int64_t E, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Kernel-path switch (test instrumentation; never needed for results).  Several stages have a specialised kernel and
 * a generic one that computes the same thing with a different mapping to the machine; a set bit forces the generic
 * kernel, so that tests/ can cross-check the two on whole full-size batches (the oracle anchors both on samples):
 *   CGTP_PATH_GENERIC_CORE   S2-S4: onsite_generic.cu instead of the lane = column core (onsite_core.cu)
 *   CGTP_PATH_GENERIC_EDGE   M3-M4: one CTA per (receiver, channel block) with direct loads (message.cu) instead of
 *                            the persistent TMA-ring kernel (edge_ring.cu)
 *   CGTP_PATH_GENERIC_PROJ   S1/S5/M1/M6: register-tiled SIMT GEMM (proj.cu) instead of proj_fast.cu / proj_multi.cu
 *   CGTP_PATH_GENERIC_SYNTH  M2: node_synth_kernel instead of the lane = column synthesis (sht_fast.cu)
 *   CGTP_PATH_UNFUSED_ONSITE S1-S5: the four-launch on-site step (projection, core per parity, projection) instead of
 *                            the single fused kernel (onsite_fused.cu)
 *   CGTP_PATH_FUSED_ONSITE   S1-S5: the single fused kernel for every shape it supports, also where the library's own
 *                            choice is the four-launch step (narrow projections N * C < 4096)
 *   CGTP_PATH_FIELD_PER_EDGE two-field coupling: one full core pass per edge and a pooling kernel (edge_field.cu) instead of
 *                            the neighbour sum on the grid inside the core (field_pool_core_kernel, onsite_core.cu)
 *   CGTP_PATH_SMEM_CORE      S2-S4 at band limits <= 6: the warp-scheduled shared-memory core (onsite_core.cu) instead of
 *                            the one-thread-per-column register core (onsite_reg.cu)
 *   CGTP_PATH_PLAIN_LAUNCH   every kernel launched in plain stream order instead of chained by programmatic dependent launch
 *                            (the kernels are the same; only their overlap at the boundaries goes away)
 * Process-wide, read at every call; 0 (default) = every specialised kernel.  CGTP_ERR_INVALID for unknown bits.
 * ------------------------------------------------------------------------------------------- */
#define CGTP_PATH_GENERIC_CORE 1
#define CGTP_PATH_GENERIC_EDGE 2
#define CGTP_PATH_GENERIC_PROJ 4
#define CGTP_PATH_GENERIC_SYNTH 8
#define CGTP_PATH_UNFUSED_ONSITE 16
#define CGTP_PATH_FUSED_ONSITE 32
#define CGTP_PATH_FIELD_PER_EDGE 64
#define CGTP_PATH_SMEM_CORE 128
#define CGTP_PATH_PLAIN_LAUNCH 256
int cgtp_set_kernel_path(int flags);
int cgtp_get_kernel_path(void);

/* ---------------------------------------------------------------------------------------------
 * FP32 pipe calibration: the denominator of the "alu" roofline of the on-site path ("measure the
 * real sustained FP32 peak with an FMA micro-benchmark on the box").  Runs a register-only kernel of dependent-chain
 * fused multiply-adds on every SM (16 independent chains per thread, 8 warps x 4 CTAs per SM) for about `ms_target`
 * milliseconds and returns the sustained rate in *tflops (2 flop per FMA lane):
 *   packed = 0  scalar FFMA (fma.rn.f32)        packed = 1  FFMA2 (fma.rn.f32x2, two lanes per instruction)
 * Synchronises `cuda_stream`.  *sm_mhz_est (may be NULL) receives flop rate / (SMs x 128 lanes x 2), the clock the
 * rate would correspond to at one FMA per lane per cycle.
 * ------------------------------------------------------------------------------------------- */
int cgtp_fma_peak(int packed, double ms_target, double* tflops, double* sm_mhz_est, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Instrumentation (used by bench.py; never needed for results).
 * cgtp_launch_count: number of kernels this library has launched since it was loaded.
 * cgtp_profile_enable(1): record a CUDA-event pair around every kernel launch (on the launching
 * stream); cgtp_profile_collect synchronises those events, adds the elapsed milliseconds and launch
 * counts per kernel kind into ms[kind], launches[kind] (arrays of cgtp_profile_kinds() entries), and
 * clears the record.  cgtp_profile_kind_name(kind) names a kind.
 * ------------------------------------------------------------------------------------------- */
int64_t cgtp_launch_count(void);
int cgtp_profile_kinds(void);
const char* cgtp_profile_kind_name(int kind);
int cgtp_profile_enable(int on);
int cgtp_profile_collect(double* ms, int64_t* launches);

#ifdef __cplusplus
}
#endif
#endif /* CGTP_H */
