// edge_field.cu -- data movement of the two-field coupling (Eq.(28) :236, Sec. VII C f
// :471): the edge side is a projected feature field a[e,c,:] that "no longer factors as R.Y", so every edge is one
// on-site product (edge field x sender field) through the fused S2-S4 core, and the per-edge rank-space results are
// pooled per receiver.  Two HBM-bound kernels around the core:
//   gather:   Hb[e][k][:] = Hn[send(e)][k][:]                  (factor 2 of Eq.(28): the sender's projected feature)
//   pool:     Tn[i][k][:] (+)= sum_{e in segment(i), e0 <= e < e1} T[e - e0][k][:]      (sum_j of Eq.(28))
// Both move whole [Cpar][stride] blocks, which are contiguous; the pooled sum runs over the receiver-sorted edges in
// edge order (fixed order, no float atomics).  Analysis is linear, so pooling the analysed coefficients equals
// analysing the pooled grid (Eq.(53)-(54) :420-:422) -- the grids themselves never leave the SM here.
#include "common.cuh"

namespace cgtp {

__global__ void __launch_bounds__(256) field_gather_kernel(const float* __restrict__ Hn, const int64_t* __restrict__ send,
                                                           float* __restrict__ Hb, long long ne, int blk,
                                                           const int32_t* __restrict__ status)
{
    if (*status != 0) return;  // senders are validated by M0; an invalid list leaves the output undefined
    for (long long e = blockIdx.x; e < ne; e += gridDim.x) {
        const float* src = Hn + (size_t)send[e] * blk;
        float* dst = Hb + (size_t)e * blk;
        if ((blk & 3) == 0) {  // 16-byte aligned blocks: 128-bit copies
            const float4* s4 = reinterpret_cast<const float4*>(src);
            float4* d4 = reinterpret_cast<float4*>(dst);
            for (int q = threadIdx.x; q < (blk >> 2); q += blockDim.x) d4[q] = __ldg(s4 + q);
            continue;
        }
        for (int q = threadIdx.x; q < blk; q += blockDim.x) dst[q] = __ldg(src + q);
    }
}

__global__ void __launch_bounds__(256) field_pool_kernel(const float* __restrict__ T, const int64_t* __restrict__ row_ptr,
                                                         float* __restrict__ Tn, long long nodes, long long e0,
                                                         long long e1, int blk, const int32_t* __restrict__ status)
{
    if (*status != 0) return;
    for (long long i = blockIdx.x; i < nodes; i += gridDim.x) {
        const long long r0 = row_ptr[i], r1 = row_ptr[i + 1];
        const long long lo = r0 > e0 ? r0 : e0, hi = r1 < e1 ? r1 : e1;
        // a segment that starts in this chunk overwrites, its continuation in later chunks adds; receivers without
        // in-edges are cleared by the first chunk (e0 == 0; the caller runs it even when there are no edges)
        const bool first = r0 >= e0;
        if (lo >= hi && !(r0 == r1 && e0 == 0)) continue;
        float* dst = Tn + (size_t)i * blk;
        if ((blk & 3) == 0) {
            // blocks of a multiple of 4 floats start 16-byte aligned (the buffers are 256-byte aligned): 128-bit loads,
            // two vectors per thread in flight; every component still adds its edges in edge order
            const float4* T4 = reinterpret_cast<const float4*>(T);
            float4* dst4 = reinterpret_cast<float4*>(dst);
            const int blk4 = blk >> 2;
            for (int q = threadIdx.x; q < blk4; q += 2 * blockDim.x) {
                const int q1 = q + blockDim.x;
                const bool two = q1 < blk4;
                float4 a0 = first ? make_float4(0.f, 0.f, 0.f, 0.f) : dst4[q];
                float4 a1 = (first || !two) ? make_float4(0.f, 0.f, 0.f, 0.f) : dst4[q1];
                for (long long e = lo; e < hi; ++e) {
                    const float4* t = T4 + (size_t)(e - e0) * blk4;
                    const float4 v0 = __ldg(t + q);
                    const float4 v1 = two ? __ldg(t + q1) : make_float4(0.f, 0.f, 0.f, 0.f);
                    a0.x += v0.x; a0.y += v0.y; a0.z += v0.z; a0.w += v0.w;
                    a1.x += v1.x; a1.y += v1.y; a1.z += v1.z; a1.w += v1.w;
                }
                dst4[q] = a0;
                if (two) dst4[q1] = a1;
            }
            continue;
        }
        for (int q = threadIdx.x; q < blk; q += blockDim.x) {
            float acc = first ? 0.f : dst[q];
            for (long long e = lo; e < hi; ++e) acc += __ldg(T + (size_t)(e - e0) * blk + q);
            dst[q] = acc;
        }
    }
}

int launch_field_gather(const float* Hn, const int64_t* send, float* Hb, int64_t ne, int blk, const int32_t* status,
                        cudaStream_t st)
{
    if (ne <= 0 || blk <= 0) return CGTP_OK;
    const int64_t grid = ne < 148 * 16 ? ne : 148 * 16;
    LaunchScope scope(K_MISC, st);
    field_gather_kernel<<<(unsigned)grid, 256, 0, st>>>(Hn, send, Hb, (long long)ne, blk, status);
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

int launch_field_pool(const float* T, const int64_t* row_ptr, float* Tn, int64_t nodes, int64_t e0, int64_t e1, int blk,
                      const int32_t* status, cudaStream_t st)
{
    if (nodes <= 0 || blk <= 0) return CGTP_OK;
    const int64_t grid = nodes < 148 * 16 ? nodes : 148 * 16;
    LaunchScope scope(K_MISC, st);
    field_pool_kernel<<<(unsigned)grid, 256, 0, st>>>(T, row_ptr, Tn, (long long)nodes, (long long)e0, (long long)e1,
                                                      blk, status);
    CGTP_CUDA_CHECK(cudaGetLastError());
    return CGTP_OK;
}

}  // namespace cgtp
