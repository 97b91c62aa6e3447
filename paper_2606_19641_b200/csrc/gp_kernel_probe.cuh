// gp_kernel_probe.cuh — calibration probes for the roofline denominators ("a tracked write-only HBM
// bandwidth and an FP32 FMA peak measured under this kernel's clock").  Not part of the render path.
#pragma once
#include "gp_device.cuh"

namespace gp {

// Write-only stream with the render pass's exact store pattern: per 128-pixel group a warp writes one 4-byte store per
// lane to the class plane and to each of the three colour planes, and one 16-byte store per lane to the instance and
// depth planes (12 bytes per pixel, full 128-byte lines).  Groups are dealt to CTAs in ascending order, 16 per CTA.
__global__ void __launch_bounds__(128, 8)
k_probe_store(size_t n_groups, uint8_t *o_cls, int32_t *o_inst, float *o_depth, uint8_t *o_rgb, size_t rgb_plane, uint32_t val) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const size_t g0 = (size_t)blockIdx.x * 16;
    for (int q = warp; q < 16; q += 4) {
        const size_t g = g0 + q;
        if (g >= n_groups) return;
        const size_t o = g * 128 + lane * 4;
        *reinterpret_cast<uint32_t *>(o_cls + o) = val;
        *reinterpret_cast<int4 *>(o_inst + o) = make_int4(-1, -1, -1, -1);
        *reinterpret_cast<float4 *>(o_depth + o) = make_float4(1.0f, 1.0f, 1.0f, 1.0f);
        // rgb is [view][3][HW]: the probe treats the whole buffer as one "view" of n pixels
        *reinterpret_cast<uint32_t *>(o_rgb + o) = val;
        *reinterpret_cast<uint32_t *>(o_rgb + rgb_plane + o) = val;
        *reinterpret_cast<uint32_t *>(o_rgb + 2 * rgb_plane + o) = val;
    }
}

// The same 12 B / pixel store stream, but with the render pass's CTA -> address mapping: one CTA of 4 warps per "view" of
// view_groups 128-pixel groups (the colour planes laid out [view][3][HW] as gp_render_batch writes them), warps taking
// strips of 4 groups in ascending order.  The CTAs resident at one time (148 x 8) then write 1184 separate windows of every
// plane instead of one compact one, which is what bounds k_render's own store stream.
__global__ void __launch_bounds__(128, 8)
k_probe_store_view(int view_groups, uint8_t *o_cls, int32_t *o_inst, float *o_depth, uint8_t *o_rgb, uint32_t val) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const size_t HW = (size_t)view_groups * 128, v0 = (size_t)blockIdx.x * HW;
    for (int q0 = warp * 4; q0 < view_groups; q0 += 16)
        for (int q = q0; q < min(q0 + 4, view_groups); ++q) {
            const size_t oi = (size_t)q * 128 + lane * 4, o = v0 + oi;
            *reinterpret_cast<uint32_t *>(o_cls + o) = val;
            *reinterpret_cast<int4 *>(o_inst + o) = make_int4(-1, -1, -1, -1);
            *reinterpret_cast<float4 *>(o_depth + o) = make_float4(1.0f, 1.0f, 1.0f, 1.0f);
            uint8_t *pr = o_rgb + 3 * v0 + oi;
            *reinterpret_cast<uint32_t *>(pr) = val;
            *reinterpret_cast<uint32_t *>(pr + HW) = val;
            *reinterpret_cast<uint32_t *>(pr + 2 * HW) = val;
        }
}

// FP32 FMA throughput: 8 independent dependent-chains of FFMA per thread, no memory traffic; out is written only if a
// result is NaN (never), which keeps the chains alive.
__global__ void __launch_bounds__(256)
k_probe_fma(int iters, float seed, float *out) {
    float a0 = seed, a1 = seed + 1.0f, a2 = seed + 2.0f, a3 = seed + 3.0f, a4 = seed + 4.0f, a5 = seed + 5.0f, a6 = seed + 6.0f,
          a7 = seed + 7.0f;
    const float m = 0.999f, c = 0.001f * (float)(threadIdx.x & 7);
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            a0 = fmaf(a0, m, c); a1 = fmaf(a1, m, c); a2 = fmaf(a2, m, c); a3 = fmaf(a3, m, c);
            a4 = fmaf(a4, m, c); a5 = fmaf(a5, m, c); a6 = fmaf(a6, m, c); a7 = fmaf(a7, m, c);
        }
    }
    const float s = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (s != s) out[0] = s;
}

// Exhaustive check of c_rcp2 against __frcp_rn: every one of the 2^32 bit patterns, each paired with a few partners
// (1, 0, 2^127, a subnormal, either sign) so that both outputs and both sides of the joint range check are exercised.
// out[0] += mismatching patterns.
__global__ void __launch_bounds__(256)
k_probe_rcp(unsigned long long *out) {
    unsigned long long bad = 0;
    const uint32_t partners[4] = {0x3f800000u, 0x00000000u, 0x7f000000u, 0x00400000u};
    for (unsigned long long b = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; b < (1ull << 32);
         b += (unsigned long long)gridDim.x * blockDim.x) {
        const float x = __uint_as_float((uint32_t)b);
        const uint32_t want = __float_as_uint(__frcp_rn(x));
        const float y = __uint_as_float(partners[b & 3] ^ (uint32_t)(b >> 7 << 31));
        const uint32_t want_y = __float_as_uint(__frcp_rn(y));
        float ix, iy;
        c_rcp2(x, y, ix, iy);
        bool ok = __float_as_uint(ix) == want && __float_as_uint(iy) == want_y;     // NaN in -> the same NaN bits out
        c_rcp2(y, x, iy, ix);
        ok = ok && __float_as_uint(ix) == want && __float_as_uint(iy) == want_y;
        if (!ok) ++bad;
    }
    for (int o = 16; o; o >>= 1) bad += __shfl_xor_sync(0xffffffffu, bad, o);
    if ((threadIdx.x & 31) == 0 && bad) atomicAdd(out, bad);
}

}  // namespace gp
