// proj_tile.cuh -- the register-tile projection of the single-kernel on-site step (onsite_fused.cu): thread tile = 4 output rows x 13 columns, packed FP32 FMAs over row pairs,
// the coefficient rows read from a raw TMA-staged block through 16-byte aligned 128-bit broadcast loads.
#pragma once

#include "sht.cuh"

namespace cgtp {

constexpr int kTM = 4;         // output rows per thread of a projection tile
constexpr int kTW = 12;        // columns per projection tile (the last tile of a row may hold 13)
constexpr int kTJ = 13;

// column tiles per row: 12 wide, the last one up to 13 (13 + 3 floats of misalignment fill the 16-float window)
__host__ __device__ inline int proj_num_slices(int L)
{
    if (L <= kTJ) return 1;
    return (L % kTW == 1) ? (L - 1) / kTW : (L + kTW - 1) / kTW;
}

__device__ __forceinline__ float4 fz_lds128(uint32_t addr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ float2 fz_lds64(uint32_t addr)
{
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}
// One contraction index of a projection tile: acc[p][t] += (w[2p], w[2p+1]) * x[t] for the thread's 4 output rows (2 packed
// pairs) and 13 columns.  x = 13 consecutive floats starting SHIFT floats after the 16-byte aligned shared-memory address
// xb (loads the compiler finds unused are dropped); the 4 weights are one 128-bit load at wb.
template <int SHIFT>
__device__ __forceinline__ void tile_fma(float2 (&acc)[2][kTJ], uint32_t xb, uint32_t wb)
{
    const float4 a = fz_lds128(xb), b = fz_lds128(xb + 16), c = fz_lds128(xb + 32), d = fz_lds128(xb + 48);
    const float v[16] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w, c.x, c.y, c.z, c.w, d.x, d.y, d.z, d.w};
    const float4 w4 = fz_lds128(wb);
    const float2 w0 = make_float2(w4.x, w4.y), w1 = make_float2(w4.z, w4.w);
#pragma unroll
    for (int t = 0; t < kTJ; ++t) {
        const float2 x = make_float2(v[SHIFT + t], v[SHIFT + t]);
        acc[0][t] = __ffma2_rn(w0, x, acc[0][t]);
        acc[1][t] = __ffma2_rn(w1, x, acc[1][t]);
    }
}

// A projection tile: acc[p][t] = sum_k W[k][rows 2p, 2p+1] * X[row k][lm0 + t].  x0 = byte address of (row 0, lm0), 16-byte
// aligned; rows are row_bytes apart.  MIS: the row stride is 1 mod 4 floats, so row k starts k mod 4 floats past a 16-byte
// boundary and the window is read from the boundary below it (static under the 4-fold unrolling); otherwise every row is
// aligned.  w0 = byte address of the thread's 4 weights of k = 0, w_kstride bytes between k.  K is a multiple of 4.
template <bool MIS>
__device__ __forceinline__ void proj_tile(float2 (&acc)[2][kTJ], uint32_t x0, uint32_t row_bytes, uint32_t w0,
                                          uint32_t w_kstride, int K)
{
#pragma unroll 2
    for (int k0 = 0; k0 < K; k0 += 4) {
        const uint32_t xb = x0 + (uint32_t)k0 * row_bytes, wb = w0 + (uint32_t)k0 * w_kstride;
        tile_fma<0>(acc, xb, wb);
        tile_fma<MIS ? 1 : 0>(acc, xb + row_bytes - (MIS ? 4u : 0u), wb + w_kstride);
        tile_fma<MIS ? 2 : 0>(acc, xb + 2 * row_bytes - (MIS ? 8u : 0u), wb + 2 * w_kstride);
        tile_fma<MIS ? 3 : 0>(acc, xb + 3 * row_bytes - (MIS ? 12u : 0u), wb + 3 * w_kstride);
    }
}

}  // namespace cgtp
