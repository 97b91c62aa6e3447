// gp_kernel_render.cuh — a3-a9: the render pass (one CTA per view).
//
//   prologue  one thread arms an mbarrier and issues two TMA bulk copies (cp.async.bulk, global ->
//             shared) of the view's list (EntryGeo n*48 B, EntryAux n*16 B); meanwhile all threads
//             build the per-column table s_j and the per-row table (v_i, d.z, 1/d.z, t_ground).
//   strips    each warp owns strips of SR consecutive rows.  It scans the list 32 entries at a time
//             (ballot on row overlap: the warp-level early-out), and for every overlapping entry
//             spreads its lanes over the entry's pixel rectangle inside the strip, runs the contract
//             slab test (C5) and keeps the lexicographic minimum (C6) as a packed 64-bit key in a
//             shared-memory key buffer that only this warp touches (no atomics).
//   resolve   per 4 consecutive pixels of a row: ground / sky default from the row table, patched by
//             the key where a primitive won; shade (C8); 4-byte / 16-byte coalesced stores: a warp
//             writes 128 consecutive pixels of every plane (full 128-byte lines).
#pragma once
#include "gp_device.cuh"

namespace gp {

struct RenderArgs {
    const ViewHdr *hdr; const EntryGeo *geo; const EntryAux *aux; const PrimMeta *meta;
    int cap, scap, world_begin, H, W;   // cap: list stride in global memory; scap: staged capacity
    float th, tv;
    int SR, log2LC;                 // rows per strip; lanes per row of the test tile (LC = 1 << log2LC)
    int log2W;                      // valid when NG > 0 (W a power of two)
    int ngr; uint32_t magicW;       // NG == 0: groups per whole strip when SR*W % 128 == 0 and W % 4 == 0 (else 0); ceil(2^32 / W)
    uint8_t *o_cls; int32_t *o_inst; float *o_depth; uint8_t *o_rgb;
    unsigned long long *stats;
    // raster variant (gp_kernel_raster.cuh): SR = rows per tile, log2W = -1 unless W is a power of two
    int ntiles;                     // tiles per view
    // divisions by launch constants, as multiplications (host side: render_device)
    int n_strips;                   // ceil(H / SR)
    uint32_t magicSR;               // ceil(2^32 / SR): row / SR = umulhi(row, magicSR) for row < 8192
    uint32_t magic_vpw; int shift_vpw;   // view / (A * C) = (view * magic_vpw) >> shift_vpw for view < 2^31
    float two_over_H, two_over_W;   // 2.0f / (float)H, 2.0f / (float)W: IEEE divisions done on the host (C2)
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n .reg .pred p;\n WAIT_%=:\n"
        " mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        " @p bra DONE_%=;\n bra WAIT_%=;\n DONE_%=:\n}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}


constexpr unsigned long long kKeyEmpty = 0xFFFFFFFFFFFFFFFFull;

// 1/x to ~1 ulp in one MUFU instruction, for the conservative (non-contract) column-interval bound of flat
// primitives only; its error is far inside the 1e-5 relative + 0.02 px slack of that bound
__device__ __forceinline__ float flat_rcp(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

// a5/a7/a8/a9 for the 4 consecutive pixels a lane owns in one 128-pixel group: ground / sky default
// from the row's t_ground, patched where a primitive's key won, then one 4-byte store per 8-bit
// plane and one 16-byte store per 32-bit plane.
__device__ __forceinline__ void resolve_quad(float tg, const uint4 *s_bg, const unsigned long long *kq,
                                             const uint32_t *__restrict__ wtab, uint8_t *pc, int32_t *pi,
                                             float *pd, uint8_t *pr, size_t HW) {
    const bool ground = tg > 0.0f;
    const uint4 bg = s_bg[ground ? 1 : 0];                 // cls4, r4, g4, b4 of the background
    uint32_t cls4 = bg.x, r4 = bg.y, g4 = bg.z, b4 = bg.w;
    int4 inst4 = make_int4(-1, -1, -1, -1);
    const float d0 = fmaxf(tg, 0.0f);                      // tg = -1 marks "no ground on this row"
    float4 dep4 = make_float4(d0, d0, d0, d0);
    if (kq) {
        const ulonglong2 ka = *reinterpret_cast<const ulonglong2 *>(kq);
        const ulonglong2 kb = *reinterpret_cast<const ulonglong2 *>(kq + 2);
        if ((ka.x & ka.y & kb.x & kb.y) != kKeyEmpty) {
#define GP_PATCH(KEY, SEL, IF, DF)                                                             \
            if ((KEY) != kKeyEmpty) {                                                          \
                const float t = __uint_as_float((uint32_t)((KEY) >> 32));                      \
                if (!ground || t <= tg) {                  /* else the ground is nearer (C6) */ \
                    const uint32_t lo = (uint32_t)(KEY);                                       \
                    const uint32_t cw = __ldg(&wtab[lo]);                                      \
                    IF = (int)__ldg(&wtab[lo | 6u]);       /* face codes are 0..5: lo|6 = slot 6 or 7 */ \
                    DF = t;                                                                    \
                    cls4 = __byte_perm(cls4, cw >> 24, SEL);                                   \
                    r4 = __byte_perm(r4, cw, SEL);                                             \
                    g4 = __byte_perm(g4, cw >> 8, SEL);                                        \
                    b4 = __byte_perm(b4, cw >> 16, SEL);                                       \
                }                                                                              \
            }
            GP_PATCH(ka.x, 0x3214, inst4.x, dep4.x)
            GP_PATCH(ka.y, 0x3240, inst4.y, dep4.y)
            GP_PATCH(kb.x, 0x3410, inst4.z, dep4.z)
            GP_PATCH(kb.y, 0x4210, inst4.w, dep4.w)
#undef GP_PATCH
        }
    }
    *reinterpret_cast<uint32_t *>(pc) = cls4;
    *reinterpret_cast<int4 *>(pi) = inst4;
    *reinterpret_cast<float4 *>(pd) = dep4;
    if (pr) {
        *reinterpret_cast<uint32_t *>(pr) = r4;
        *reinterpret_cast<uint32_t *>(pr + HW) = g4;
        *reinterpret_cast<uint32_t *>(pr + 2 * HW) = b4;
    }
}

// The same for 4 consecutive pixels that straddle two image rows (W % 4 != 0): the first `nsplit`
// pixels lie on the row with ground depth tga, the others on the next row (tgb).
__device__ __forceinline__ void resolve_quad_split(float tga, float tgb, int nsplit, const uint4 *s_bg,
                                                   const unsigned long long *kq, const uint32_t *__restrict__ wtab,
                                                   uint8_t *pc, int32_t *pi, float *pd, uint8_t *pr, size_t HW) {
    float tgv[4];
    uint32_t m = 0;                                        // byte mask of the pixels whose background is ground
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        tgv[e] = e < nsplit ? tga : tgb;
        if (tgv[e] > 0.0f) m |= 0xffu << (8 * e);
    }
    const uint4 sky = s_bg[0], gnd = s_bg[1];
    uint32_t cls4 = (gnd.x & m) | (sky.x & ~m), r4 = (gnd.y & m) | (sky.y & ~m);
    uint32_t g4 = (gnd.z & m) | (sky.z & ~m), b4 = (gnd.w & m) | (sky.w & ~m);
    int4 inst4 = make_int4(-1, -1, -1, -1);
    float4 dep4 = make_float4(fmaxf(tgv[0], 0.0f), fmaxf(tgv[1], 0.0f), fmaxf(tgv[2], 0.0f), fmaxf(tgv[3], 0.0f));
    if (kq) {
        const ulonglong2 ka = *reinterpret_cast<const ulonglong2 *>(kq);
        const ulonglong2 kb = *reinterpret_cast<const ulonglong2 *>(kq + 2);
        if ((ka.x & ka.y & kb.x & kb.y) != kKeyEmpty) {
#define GP_PATCH(KEY, E, SEL, IF, DF)                                                          \
            if ((KEY) != kKeyEmpty) {                                                          \
                const float t = __uint_as_float((uint32_t)((KEY) >> 32));                      \
                if (!(tgv[E] > 0.0f) || t <= tgv[E]) {     /* else the ground is nearer (C6) */ \
                    const uint32_t lo = (uint32_t)(KEY);                                       \
                    const uint32_t cw = __ldg(&wtab[lo]);                                      \
                    IF = (int)__ldg(&wtab[lo | 6u]);                                           \
                    DF = t;                                                                    \
                    cls4 = __byte_perm(cls4, cw >> 24, SEL);                                   \
                    r4 = __byte_perm(r4, cw, SEL);                                             \
                    g4 = __byte_perm(g4, cw >> 8, SEL);                                        \
                    b4 = __byte_perm(b4, cw >> 16, SEL);                                       \
                }                                                                              \
            }
            GP_PATCH(ka.x, 0, 0x3214, inst4.x, dep4.x)
            GP_PATCH(ka.y, 1, 0x3240, inst4.y, dep4.y)
            GP_PATCH(kb.x, 2, 0x3410, inst4.z, dep4.z)
            GP_PATCH(kb.y, 3, 0x4210, inst4.w, dep4.w)
#undef GP_PATCH
        }
    }
    *reinterpret_cast<uint32_t *>(pc) = cls4;
    *reinterpret_cast<int4 *>(pi) = inst4;
    *reinterpret_cast<float4 *>(pd) = dep4;
    if (pr) {
        *reinterpret_cast<uint32_t *>(pr) = r4;
        *reinterpret_cast<uint32_t *>(pr + HW) = g4;
        *reinterpret_cast<uint32_t *>(pr + 2 * HW) = b4;
    }
}

// Contract C5 (per-pixel part) + C6 for one ray against one staged entry: exact fp32 slab test and
// lexicographic-minimum update of the pixel's key.  g0 = (ax bx ay by); dlx, dly are the box-frame direction
// (already formed with the contract's fma chain); (loz, hiz) is the z slab interval, which depends on the row
// only and is formed once per row by slab_z; dz is the row's d.z.
__device__ __forceinline__ void slab_z(const float4 &g1, const float4 &rt, float &loz, float &hiz) {
    const float ta = c_mul(g1.x, rt.z), tb = c_mul(g1.y, rt.z);
    loz = c_min(ta, tb); hiz = c_max(ta, tb);
}
template <bool ATOMIC>      // ATOMIC: other lanes of the warp may update the same key at the same time
__device__ __forceinline__ void slab_select(const float4 &g0, float dlx, float dly, float loz, float hiz, float dz,
                                            float t_max, bool flat, uint32_t klow, unsigned long long *kp) {
    float ix, iy;
    c_rcp2(dlx, dly, ix, iy);                          // == c_rcp(dlx), c_rcp(dly)
    float ta, tb;
    ta = c_mul(g0.x, ix); tb = c_mul(g0.y, ix);
    const float lox = c_min(ta, tb), hix = c_max(ta, tb);
    ta = c_mul(g0.z, iy); tb = c_mul(g0.w, iy);
    const float loy = c_min(ta, tb), hiy = c_max(ta, tb);
    const float tn = c_max(c_max(lox, loy), loz);
    const float tf = c_min(c_min(hix, hiy), hiz);
    if (tn <= tf && tn > 0.0f && tn <= t_max) {
        uint32_t face;                                  // m*2 + (sigma > 0)
        if (flat) face = 5;
        else if (lox == tn) face = 0 + (dlx > 0.0f ? 0 : 1);
        else if (loy == tn) face = 2 + (dly > 0.0f ? 0 : 1);
        else face = 4 + (dz > 0.0f ? 0 : 1);
        const unsigned long long key = ((unsigned long long)__float_as_uint(tn) << 32) | klow | face;   // C6
        if (key < *kp) {                                // (racy pre-read under ATOMIC: keys only ever decrease)
            if (ATOMIC) atomicMin(kp, key);
            else *kp = key;
        }
    }
}

// ---- a6 / a7 for one strip -------------------------------------------------------------------------
constexpr int kOverlapCap = 64;      // entries of one strip worked off per batch (per-warp overlap list)
#ifndef GP_SHORT_SPAN
#define GP_SHORT_SPAN 3
#endif
constexpr int kShortSpan = GP_SHORT_SPAN;   // flat-quad column spans up to this many pixels are finished by their own lane

struct StripBatchCtx {
    const EntryGeo *s_geo, *g_geo; const EntryAux *s_aux, *g_aux;
    const float4 *s_row; const float *s_col;
    int scap, W, log2LC;
    float th, t_max;
};
struct EntryRec { float4 g0, g1, g2; uint4 ax; };   // (ax bx ay by) (az bz flx fly) (rlx rly ulx uly) aux

__device__ __forceinline__ EntryRec load_entry(const StripBatchCtx &c, int eb) {
    EntryRec r;
    if (eb < c.scap) {
        const float4 *sg = reinterpret_cast<const float4 *>(&c.s_geo[eb]);
        r.g0 = sg[0]; r.g1 = sg[1]; r.g2 = sg[2];
        r.ax = *reinterpret_cast<const uint4 *>(&c.s_aux[eb]);
    } else {                            // rare: list longer than the staged capacity
        const float4 *gg = reinterpret_cast<const float4 *>(&c.g_geo[eb]);
        r.g0 = __ldg(gg); r.g1 = __ldg(gg + 1); r.g2 = __ldg(gg + 2);
        r.ax = __ldg(reinterpret_cast<const uint4 *>(&c.g_aux[eb]));
    }
    return r;
}

// Conservative column interval [ja, jb] of a flat entry on one image row (not contract arithmetic: plain fp32 +
// slack): the plane depth t is fixed per row, so the footprint of the quad on that row is one interval.
// flat_prepare: the part that depends on the entry only; flat_row: one row.
struct FlatBound { float mx, my, hxs, hys, col_scale, halfW; };
__device__ __forceinline__ FlatBound flat_prepare(const float4 &g0, const float4 &g1, int W, float th) {
    FlatBound fb;
    // centre -ol and half extents h in the ray-origin frame, recovered from a = -h - ol, b = h - ol
    fb.mx = 0.5f * (g0.x + g0.y); fb.my = 0.5f * (g0.z + g0.w);
    const float mz = 0.5f * (g1.x + g1.y);
    const float ex_ = 0.5f * (g0.y - g0.x), ey_ = 0.5f * (g0.w - g0.z);
    const float dl_ = 2e-5f * (fabsf(fb.mx) + fabsf(fb.my) + fabsf(mz) + ex_ + ey_) + 1e-6f;
    fb.hxs = ex_ + dl_; fb.hys = ey_ + dl_;
    fb.col_scale = 0.5f * (float)W / th; fb.halfW = 0.5f * (float)W;
    return fb;
}
__device__ __forceinline__ void flat_row(const FlatBound &fb, const float4 &g1, const float4 &g2, const float4 &rt,
                                         float t_max, int W, int c0, int c1, int &ja, int &jb) {
    ja = 1; jb = 0;
    const float t = g1.x * rt.z;                     // plane depth on this row
    if (!(t > 0.0f && t <= t_max * 1.00001f)) return;
    const float X0 = fmaf(t, fmaf(rt.x, g2.z, g1.z), -fb.mx), X1 = t * g2.x;
    const float Y0 = fmaf(t, fmaf(rt.x, g2.w, g1.w), -fb.my), Y1 = t * g2.y;
    float slo = -3.0e38f, shi = 3.0e38f;
    bool ok = true;
    if (fabsf(X1) > 1e-12f) {
        const float r = flat_rcp(X1), a = (-fb.hxs - X0) * r, b = (fb.hxs - X0) * r;
        slo = fmaxf(slo, fminf(a, b)); shi = fminf(shi, fmaxf(a, b));
    } else ok = fabsf(X0) <= fb.hxs;
    if (fabsf(Y1) > 1e-12f) {
        const float r = flat_rcp(Y1), a = (-fb.hys - Y0) * r, b = (fb.hys - Y0) * r;
        slo = fmaxf(slo, fminf(a, b)); shi = fminf(shi, fmaxf(a, b));
    } else ok = ok && fabsf(Y0) <= fb.hys;
    if (!(ok && slo <= shi)) return;
    // column of s: (s/th + 1) W/2 - 0.5, widened by 0.02 px + relative slack
    const float xa = fmaf(slo, fb.col_scale, fb.halfW - 0.52f) - 1e-5f * fabsf(slo * fb.col_scale);
    const float xb = fmaf(shi, fb.col_scale, fb.halfW - 0.48f) + 1e-5f * fabsf(shi * fb.col_scale);
    ja = max(c0, (int)ceilf(fmaxf(xa, -1.0f)));
    jb = min(c1, (int)floorf(fminf(xb, (float)W)));
}
__device__ __forceinline__ void flat_interval(const EntryRec &E, const float4 &rt, const StripBatchCtx &c, int &ja, int &jb) {
    const FlatBound fb = flat_prepare(E.g0, E.g1, c.W, c.th);
    flat_row(fb, E.g1, E.g2, rt, c.t_max, c.W, (int)(E.ax.z & 0xffff), (int)(E.ax.z >> 16), ja, jb);
}

// The gathered entries of one strip: olist[0 .. nfl) flat quads, olist[kOverlapCap - nbx .. kOverlapCap) boxes and
// spheres.  Flat quads: one lane per (entry, row) bounds the row's column interval; a short interval is finished
// by that lane (atomic minimum: two lanes may meet on a pixel), a long one is spread over the warp afterwards.
// Boxes / spheres: the warp spreads over the entry's pixel rectangle inside the strip.  Returns the number of
// exact tests (STATS only).
template <bool STATS, bool SPH>
__device__ __forceinline__ unsigned strip_batch(const StripBatchCtx &c, const uint16_t *olist, int nfl, int nbx,
                                                int row0, int row1, unsigned long long *keys, int lane) {
    unsigned n_tests = 0;
    const int W = c.W;
    const float t_max = c.t_max;
    const int nrows = row1 - row0 + 1;
    // ---- flat quads -------------------------------------------------------------------------------
    const int nitems = nfl * nrows;
    const bool pow2 = (nrows & (nrows - 1)) == 0;             // rows per strip: a power of two except in a ragged last strip
    const int sh = 31 - __clz(nrows);
    for (int t0 = 0; t0 < nitems; t0 += 32) {
        const int t = t0 + lane;
        int ja = 1, jb = 0, i = row0, eb = 0;
        uint32_t klow = 0;
        if (t < nitems) {
            const int le = pow2 ? t >> sh : t / nrows;
            i = row0 + (t - le * nrows);
            eb = olist[le];
            const EntryRec E = load_entry(c, eb);
            klow = (E.ax.x >> 2) << 3;
            if (i >= (int)(E.ax.y & 0xffff) && i <= (int)(E.ax.y >> 16)) {
                const float4 rt = c.s_row[i];
                const int c0 = (int)(E.ax.z & 0xffff), c1 = (int)(E.ax.z >> 16);
                if (c1 - c0 < kShortSpan) { ja = c0; jb = c1; }    // a few columns only: not worth bounding further
                else flat_interval(E, rt, c, ja, jb);
                if (jb - ja < kShortSpan) {                        // short (or empty): finish it here
                    float loz, hiz;
                    slab_z(E.g1, rt, loz, hiz);
                    unsigned long long *krow = keys + (i - row0) * W;
                    for (int j = ja; j <= jb; ++j) {
                        if (STATS) ++n_tests;
                        const float s = c.s_col[j];
                        const float dlx = c_fma(rt.x, E.g2.z, c_fma(s, E.g2.x, E.g1.z));
                        const float dly = c_fma(rt.x, E.g2.w, c_fma(s, E.g2.y, E.g1.w));
                        slab_select<true>(E.g0, dlx, dly, loz, hiz, rt.y, t_max, true, klow, krow + j);
                    }
                    jb = ja - 1;                                   // done
                }
            }
        }
        __syncwarp();
        unsigned lm = __ballot_sync(0xffffffffu, jb >= ja);        // long spans: all lanes, one item at a time
        while (lm) {
            const int src = __ffs(lm) - 1;
            lm &= lm - 1;
            const int bi = __shfl_sync(0xffffffffu, i, src), beb = __shfl_sync(0xffffffffu, eb, src);
            const int bja = __shfl_sync(0xffffffffu, ja, src), bjb = __shfl_sync(0xffffffffu, jb, src);
            const EntryRec E = load_entry(c, beb);
            const uint32_t bk = (E.ax.x >> 2) << 3;
            const float4 rt = c.s_row[bi];
            float loz, hiz;
            slab_z(E.g1, rt, loz, hiz);
            unsigned long long *krow = keys + (bi - row0) * W;
            for (int j = bja + lane; j <= bjb; j += 32) {
                if (STATS) ++n_tests;
                const float s = c.s_col[j];
                const float dlx = c_fma(rt.x, E.g2.z, c_fma(s, E.g2.x, E.g1.z));
                const float dly = c_fma(rt.x, E.g2.w, c_fma(s, E.g2.y, E.g1.w));
                slab_select<false>(E.g0, dlx, dly, loz, hiz, rt.y, t_max, true, bk, krow + j);
            }
            __syncwarp();
        }
    }
    // ---- boxes and spheres ------------------------------------------------------------------------
    const int LC = 1 << c.log2LC, LR = 32 >> c.log2LC;
    const int li = lane >> c.log2LC, lj = lane & (LC - 1);
    for (int ib = 0; ib < nbx; ++ib) {
        const EntryRec E = load_entry(c, olist[kOverlapCap - 1 - ib]);
        const float4 &g0 = E.g0, &g1 = E.g1, &g2 = E.g2;
        const uint32_t kind = E.ax.x & 3u, klow = (E.ax.x >> 2) << 3;
        const int r0 = max((int)(E.ax.y & 0xffff), row0), r1 = min((int)(E.ax.y >> 16), row1);
        const int c0 = (int)(E.ax.z & 0xffff), c1 = (int)(E.ax.z >> 16);
        for (int rb = r0; rb <= r1; rb += LR) {
            const int i = min(rb + li, r1);                         // lanes past r1 idle (j loop below)
            const bool row_ok = rb + li <= r1;
            const float4 rt = c.s_row[i];                           // v, dz, 1/dz, tg
            unsigned long long *krow = keys + (i - row0) * W;
            if (SPH && kind == kKindSphere) {
                // C5s over the entry's pixel rectangle; g0 = (e.x, e.y, e.z, r*r), basis = world frame
                for (int cb = c0; cb <= c1; cb += LC) {
                    const int j = cb + lj;
                    if (row_ok && j <= c1) {
                        if (STATS) ++n_tests;
                        const float s = c.s_col[j];
                        const float dx = c_fma(rt.x, g2.z, c_fma(s, g2.x, g1.z));
                        const float dy = c_fma(rt.x, g2.w, c_fma(s, g2.y, g1.w));
                        const float tn = sphere_entry(g0.x, g0.y, g0.z, g0.w, dx, dy, rt.y);
                        if (tn > 0.0f && tn <= t_max) {
                            const unsigned long long key = ((unsigned long long)__float_as_uint(tn) << 32) | klow | 5u;
                            if (key < krow[j]) krow[j] = key;
                        }
                    }
                }
            } else {
                float loz, hiz;
                slab_z(g1, rt, loz, hiz);                           // per row, not per pixel
                for (int cb = c0; cb <= c1; cb += LC) {
                    const int j = cb + lj;
                    if (row_ok && j <= c1) {
                        if (STATS) ++n_tests;
                        const float s = c.s_col[j];
                        const float dlx = c_fma(rt.x, g2.z, c_fma(s, g2.x, g1.z));      // C5, per-pixel part
                        const float dly = c_fma(rt.x, g2.w, c_fma(s, g2.y, g1.w));
                        slab_select<false>(g0, dlx, dly, loz, hiz, rt.y, t_max, false, klow, krow + j);
                    }
                }
            }
        }
        __syncwarp();
    }
    return n_tests;
}

#ifndef GP_RENDER_WARPS
#define GP_RENDER_WARPS 4          // warps per CTA (one CTA per view)
#endif
#ifndef GP_RENDER_MIN_CTAS
#define GP_RENDER_MIN_CTAS (32 / GP_RENDER_WARPS)
#endif
// NG: 128-pixel groups per strip when W is a power of two (1, 2, 4), else 0.  SPH: the scene holds spheres
// (scenes without any run the variant compiled without the C5s branch: it costs the strip loop registers).
// GATHER: how a strip works off its list.  true: the overlapping entries are first gathered into a per-warp list and
// flat quads get one lane per (entry, row) (fewer instructions when many entries meet a strip: small images, dense
// scenes); false: entry by entry as the ballot finds them, the warp spread over each entry's rectangle (1 % faster
// when lists are short and the kernel is store-bound).  The host picks (gp_lib.cu).
#ifndef GP_RENDER_DYNAMIC
#define GP_RENDER_DYNAMIC 1
#endif
template <bool STATS, int NG, bool SPH, bool GATHER>
__global__ void __launch_bounds__(GP_RENDER_WARPS * 32, GP_RENDER_MIN_CTAS)
k_render(SceneConst sc, RenderArgs ra) {
    constexpr bool DYN = GP_RENDER_DYNAMIC != 0;
    extern __shared__ __align__(16) unsigned char smem[];
    const int view = blockIdx.x;
    const int H = ra.H, W = ra.W, SR = ra.SR;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    // ---- shared memory carve-up ---------------------------------------------------------------
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem);
    uint4 *s_bg = reinterpret_cast<uint4 *>(smem + 16);            // [0] sky, [1] ground: cls4, r4, g4, b4
    EntryGeo *s_geo = reinterpret_cast<EntryGeo *>(smem + 48);
    EntryAux *s_aux = reinterpret_cast<EntryAux *>(smem + 48 + (size_t)ra.scap * 48);
    float4 *s_row = reinterpret_cast<float4 *>(smem + 48 + (size_t)ra.scap * 64);
    float *s_col = reinterpret_cast<float *>(s_row + H);
    uint16_t *s_olist = reinterpret_cast<uint16_t *>(s_col + ((W + 3) & ~3));          // [warps][kOverlapCap], GATHER only
    unsigned long long *s_keys = reinterpret_cast<unsigned long long *>(s_olist + (GATHER ? (blockDim.x >> 5) * kOverlapCap : 0));
    unsigned long long *keys = s_keys + (size_t)warp * SR * W;

    // ---- view-independent part of the prologue (runs ahead of the cull's last CTAs under programmatic dependent launch) ----
    int *s_next = reinterpret_cast<int *>(smem + 8);               // dynamic strip counter
    if (threadIdx.x == 32 % blockDim.x) {
        const uint32_t g = shade_rgb(sc.pal[1], shade_scale(c_max(sc.Lz, 0.0f), sc.ambient)), k = sc.pal[0];
        s_bg[0] = make_uint4(0u, (k & 0xff) * 0x01010101u, ((k >> 8) & 0xff) * 0x01010101u, ((k >> 16) & 0xff) * 0x01010101u);
        s_bg[1] = make_uint4(0x01010101u, (g & 0xff) * 0x01010101u, ((g >> 8) & 0xff) * 0x01010101u,
                             ((g >> 16) & 0xff) * 0x01010101u);
    }
    if (threadIdx.x == 0) {
        *s_next = 0;
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // column table (contract C2; 2 / W and 2 / H are IEEE divisions done once on the host: the same fp32 numbers pix_s /
    // pix_v form)
    for (int j = threadIdx.x; j < W; j += blockDim.x)
        s_col[j] = c_mul(c_sub(c_mul(c_add((float)j, 0.5f), ra.two_over_W), 1.0f), ra.th);
#if GP_PDL
    // Programmatic dependent launch: wait for the cull's grid before the first read of what it wrote (returns at once when
    // the kernel was launched normally).
    asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
    const float4 vh4 = __ldg(reinterpret_cast<const float4 *>(&ra.hdr[view]));
    ViewHdr vh; vh.n = __float_as_int(vh4.x); vh.oz = vh4.y; vh.cp = vh4.z; vh.sp = vh4.w;
    const int n = vh.n & 0x7ffff, rmin = (int)((uint32_t)vh.n >> 19);
    if (threadIdx.x == 0 && n > 0) {
        const uint32_t ns = (uint32_t)min(n, ra.scap);       // entries beyond scap are read from global memory
        mbar_expect_tx(bar, ns * 64u);
        bulk_g2s(s_geo, ra.geo + (size_t)view * ra.cap, ns * 48u, bar);
        bulk_g2s(s_aux, ra.aux + (size_t)view * ra.cap, ns * 16u, bar);
    }
    // row table (contract C3-C4), overlapped with the bulk copies
    for (int i = threadIdx.x; i < H; i += blockDim.x) {
        const float v = c_mul(c_sub(1.0f, c_mul(c_add((float)i, 0.5f), ra.two_over_H)), ra.tv);
        const float dz = c_fma(v, vh.cp, vh.sp);
        const float inv_z = c_rcp(dz);
        float tg = -1.0f;
        if (dz < 0.0f) {
            const float t = c_mul(c_sub(0.0f, vh.oz), inv_z);
            if (t > 0.0f && t <= sc.t_max) tg = t;
        }
        s_row[i] = make_float4(v, dz, inv_z, tg);
    }
    __syncthreads();                       // tables + mbarrier init visible

    const int w = ra.world_begin + (int)(((unsigned long long)(unsigned)view * ra.magic_vpw) >> ra.shift_vpw);   // view / (A C)
    const uint32_t *wtab = reinterpret_cast<const uint32_t *>(ra.meta + (size_t)w * sc.P);   // uint32[P][8]
    const size_t HW = (size_t)H * W;
    const int n_strips = ra.n_strips;
    // resolve pass: lane owns pixels 4*lane .. 4*lane+3 of every 128-pixel group of the strip
    const int lane_row = (lane * 4) / W, lane_col = (lane * 4) % W;
    const int step_row = 128 / W, step_col = 128 % W;
    unsigned long long n_tests = 0;

    // Strip schedule: strips are handed out dynamically in ascending order (ascending addresses are
    // also what the HBM likes: a descending order measured 13% slower).  Strips wholly above the first
    // row any entry touches need no list and are rendered while the bulk copies are still in flight.
    const int n_free = n > 0 ? min(n_strips, (int)__umulhi((unsigned)rmin, ra.magicSR)) : n_strips;    // rmin / SR
    const EntryGeo *g_geo = ra.geo + (size_t)view * ra.cap;
    const EntryAux *g_aux = ra.aux + (size_t)view * ra.cap;
    bool list_ready = false;
    const int n_warps = blockDim.x >> 5;
    for (int strip_it = warp;; strip_it += n_warps) {
        int strip = strip_it;
        if (DYN) {                                                      // dynamic hand-out (balances long lists)
            // (plain PTX: nvcc wraps atomicAdd in a warp-aggregation sequence of ~15 instructions, for one lane)
            if (lane == 0) asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(strip) : "r"(smem_u32(s_next)) : "memory");
            strip = __shfl_sync(0xffffffffu, strip, 0);
        }
        if (strip >= n_strips) break;
        if (strip >= n_free && !list_ready) { mbar_wait(bar, 0); list_ready = true; }
        const int nn = strip < n_free ? 0 : n;                      // entries to scan for this strip
        const int row0 = strip * SR, row1 = min(H, row0 + SR) - 1;
        bool any = false;
        if (GATHER) {
            const unsigned lt_mask = (1u << lane) - 1u;
            uint16_t *olist = s_olist + warp * kOverlapCap;
            StripBatchCtx sb;
            sb.s_geo = s_geo; sb.g_geo = g_geo; sb.s_aux = s_aux; sb.g_aux = g_aux;
            sb.s_row = s_row; sb.s_col = s_col; sb.scap = ra.scap; sb.W = W; sb.log2LC = ra.log2LC; sb.th = ra.th; sb.t_max = sc.t_max;
            // ---- a3: warp-level early-out over the list: the entries whose rows overlap the strip are gathered
            // (ballot) into the warp's overlap list, flat quads from the front, boxes / spheres from the back;
            // a6/a7 then run per batch in strip_batch().
            int nfl = 0, nbx = 0;
            for (int base = 0; base < nn; base += 32) {
                const int e = base + lane;
                bool ov = false, fl = false;
                if (e < nn) {
                    const uint2 kr = e < ra.scap ? *reinterpret_cast<const uint2 *>(&s_aux[e])
                                                 : __ldg(reinterpret_cast<const uint2 *>(&g_aux[e]));   // kf, rows
                    ov = (int)(kr.y & 0xffff) <= row1 && (int)(kr.y >> 16) >= row0;
                    fl = (kr.x & 3u) == kKindFlat;
                }
                const unsigned fmask = __ballot_sync(0xffffffffu, ov && fl), bmask = __ballot_sync(0xffffffffu, ov && !fl);
                if (!(fmask | bmask)) continue;
                if (!any) {
                    any = true;
                    ulonglong2 *k2 = reinterpret_cast<ulonglong2 *>(keys);
                    const int nk2 = (row1 - row0 + 1) * W / 2;
                    for (int q = lane; q < nk2; q += 32) k2[q] = make_ulonglong2(kKeyEmpty, kKeyEmpty);
                }
                if (nfl + nbx + __popc(fmask) + __popc(bmask) > kOverlapCap) {       // no room: work off what is gathered
                    __syncwarp();
                    n_tests += strip_batch<STATS, SPH>(sb, olist, nfl, nbx, row0, row1, keys, lane);
                    nfl = nbx = 0;
                }
                if (ov && fl) olist[nfl + __popc(fmask & lt_mask)] = (uint16_t)e;
                if (ov && !fl) olist[kOverlapCap - 1 - (nbx + __popc(bmask & lt_mask))] = (uint16_t)e;
                nfl += __popc(fmask); nbx += __popc(bmask);
            }
            if (nfl + nbx) {
                __syncwarp();
                n_tests += strip_batch<STATS, SPH>(sb, olist, nfl, nbx, row0, row1, keys, lane);
            }
        } else {
            const int LC = 1 << ra.log2LC, LR = 32 >> ra.log2LC;
            const int li = lane >> ra.log2LC, lj = lane & (LC - 1);
            const float t_max = sc.t_max;
            // ---- a3: warp-level early-out over the list, a6/a7: slab test + select ----------------
            for (int base = 0; base < nn; base += 32) {
                const int e = base + lane;
                bool ov = false;
                if (e < nn) {
                    const uint32_t rows = e < ra.scap ? s_aux[e].rows : __ldg(&g_aux[e].rows);
                    ov = (int)(rows & 0xffff) <= row1 && (int)(rows >> 16) >= row0;
                }
                unsigned mask = __ballot_sync(0xffffffffu, ov);
                if (mask && !any) {
                    any = true;
                    ulonglong2 *k2 = reinterpret_cast<ulonglong2 *>(keys);
                    const int nk2 = (row1 - row0 + 1) * W / 2;
                    for (int q = lane; q < nk2; q += 32) k2[q] = make_ulonglong2(kKeyEmpty, kKeyEmpty);
                    __syncwarp();
                }
                while (mask) {
                    const int eb = base + __ffs(mask) - 1;
                    mask &= mask - 1;
                    float4 g0, g1, g2; uint4 ax;        // (ax bx ay by) (az bz flx fly) (rlx rly ulx uly) aux
                    if (eb < ra.scap) {
                        const float4 *sg = reinterpret_cast<const float4 *>(&s_geo[eb]);
                        g0 = sg[0]; g1 = sg[1]; g2 = sg[2];
                        ax = *reinterpret_cast<const uint4 *>(&s_aux[eb]);
                    } else {                            // rare: list longer than the staged capacity
                        const float4 *gg = reinterpret_cast<const float4 *>(&g_geo[eb]);
                        g0 = __ldg(gg); g1 = __ldg(gg + 1); g2 = __ldg(gg + 2);
                        ax = __ldg(reinterpret_cast<const uint4 *>(&g_aux[eb]));
                    }
                    const uint32_t kind = ax.x & 3u;
                    const bool flat = kind == kKindFlat;
                    const uint32_t klow = (ax.x >> 2) << 3;
                    const int r0 = max((int)(ax.y & 0xffff), row0), r1 = min((int)(ax.y >> 16), row1);
                    const int c0 = (int)(ax.z & 0xffff), c1 = (int)(ax.z >> 16);
                    if (SPH && kind == kKindSphere) {
                        // C5s over the entry's pixel rectangle; g0 = (e.x, e.y, e.z, r*r), basis = world frame
                        for (int rb = r0; rb <= r1; rb += LR) {
                            const int i = rb + li;
                            for (int cb = c0; cb <= c1; cb += LC) {
                                const int j = cb + lj;
                                if (i <= r1 && j <= c1) {
                                    if (STATS) ++n_tests;
                                    const float s = s_col[j];
                                    const float4 rt = s_row[i];
                                    const float dx = c_fma(rt.x, g2.z, c_fma(s, g2.x, g1.z));
                                    const float dy = c_fma(rt.x, g2.w, c_fma(s, g2.y, g1.w));
                                    const float tn = sphere_entry(g0.x, g0.y, g0.z, g0.w, dx, dy, rt.y);
                                    if (tn > 0.0f && tn <= t_max) {
                                        const unsigned long long key = ((unsigned long long)__float_as_uint(tn) << 32) | klow | 5u;
                                        unsigned long long *kp = &keys[(i - row0) * W + j];
                                        if (key < *kp) *kp = key;
                                    }
                                }
                            }
                        }
                    } else if (flat && c1 - c0 >= LC) {
                        // Wide flat primitive: per row, the plane depth t is fixed, so the footprint is one
                        // column interval.  Bound it conservatively (plain fp32 + slack) and run the exact
                        // test only inside it: a thin diagonal marking costs ~its length, not its bbox area.
                        const FlatBound fb = flat_prepare(g0, g1, W, ra.th);       // conservative bound, not contract arithmetic
                        for (int rb = r0; rb <= r1; rb += LR) {
                            const int i = rb + li;
                            int ja = 1, jb = 0;                                  // empty
                            float4 rt = make_float4(0.f, 0.f, 0.f, 0.f);
                            if (i <= r1) {
                                rt = s_row[i];
                                flat_row(fb, g1, g2, rt, t_max, W, c0, c1, ja, jb);
                            }
                            float loz, hiz;
                            slab_z(g1, rt, loz, hiz);
                            unsigned long long *krow = keys + (i - row0) * W;
                            for (int j = ja + lj; __any_sync(0xffffffffu, j <= jb); j += LC) {
                                if (j <= jb) {
                                    if (STATS) ++n_tests;
                                    const float s = s_col[j];
                                    const float dlx = c_fma(rt.x, g2.z, c_fma(s, g2.x, g1.z));
                                    const float dly = c_fma(rt.x, g2.w, c_fma(s, g2.y, g1.w));
                                    slab_select<false>(g0, dlx, dly, loz, hiz, rt.y, t_max, true, klow, krow + j);
                                }
                            }
                        }
                    } else {
                        for (int rb = r0; rb <= r1; rb += LR) {
                            const int i = min(rb + li, r1);                         // lanes past r1 idle (j loop below)
                            const bool row_ok = rb + li <= r1;
                            const float4 rt = s_row[i];                             // v, dz, 1/dz, tg
                            float loz, hiz;
                            slab_z(g1, rt, loz, hiz);                               // per row, not per pixel
                            unsigned long long *krow = keys + (i - row0) * W;
                            for (int cb = c0; cb <= c1; cb += LC) {
                                const int j = cb + lj;
                                if (row_ok && j <= c1) {
                                    if (STATS) ++n_tests;
                                    const float s = s_col[j];
                                    const float dlx = c_fma(rt.x, g2.z, c_fma(s, g2.x, g1.z));
                                    const float dly = c_fma(rt.x, g2.w, c_fma(s, g2.y, g1.w));
                                    slab_select<false>(g0, dlx, dly, loz, hiz, rt.y, t_max, flat, klow, krow + j);
                                }
                            }
                        }
                    }
                    __syncwarp();
                }
            }
        }
        // ---- a5 ground, a7 resolve, a8 shade, a9 store: 4 consecutive pixels per lane ----------
        {
            const size_t o0 = (size_t)view * HW + (size_t)row0 * W + lane * 4;
            uint8_t *pc = ra.o_cls + o0;
            int32_t *pi = ra.o_inst + o0;
            float *pd = ra.o_depth + o0;
            uint8_t *pr = ra.o_rgb ? ra.o_rgb + 2 * (size_t)view * HW + o0 : nullptr;
            const unsigned long long *kq = any ? keys + lane * 4 : nullptr;
            if (NG > 0) {       // strip = NG groups of 128 pixels, W a power of two: constant offsets
#pragma unroll
                for (int it = 0; it < NG; ++it) {
                    const int row = row0 + ((lane * 4 + it * 128) >> ra.log2W);
                    resolve_quad(s_row[row].w, s_bg, kq ? kq + it * 128 : nullptr, wtab, pc + it * 128,
                                 pi + it * 128, pd + it * 128, pr ? pr + it * 128 : nullptr, HW);
                }
            } else if (ra.ngr > 0 && row1 - row0 + 1 == SR) {
                // W % 4 == 0 and the strip is a whole number of 128-pixel groups (e.g. 96 x 4, 192 x 2, 112 x 8):
                // no row straddling, no ragged tail; the row of a pixel by a multiply-high with ceil(2^32 / W)
                for (int it = 0; it < ra.ngr; ++it) {
                    const int off = it * 128;
                    const int row = row0 + (int)__umulhi((unsigned)(lane * 4 + off), ra.magicW);
                    resolve_quad(s_row[row].w, s_bg, kq ? kq + off : nullptr, wtab, pc + off, pi + off, pd + off,
                                 pr ? pr + off : nullptr, HW);
                }
            } else {
                // any W: the strip is SR*W consecutive pixels (a multiple of 4, start 4-aligned); a lane's
                // 4 pixels straddle two rows only when W % 4 != 0, and then every lane takes the per-pixel-row form: a warp
                // in which one lane straddles would otherwise run both forms (210 x 126: 4.17 -> 4.05 ms)
                int row = row0 + lane_row, col = lane_col, off = 0;
                while (row <= row1) {
                    if ((W & 3) == 0)
                        resolve_quad(s_row[row].w, s_bg, kq ? kq + off : nullptr, wtab, pc + off, pi + off, pd + off,
                                     pr ? pr + off : nullptr, HW);
                    else {      // one code path for the warp: nsplit = 4 for the lanes that do not straddle
                        const int nsplit = min(4, W - col);
                        resolve_quad_split(s_row[row].w, s_row[row + (nsplit < 4)].w, nsplit, s_bg, kq ? kq + off : nullptr, wtab,
                                           pc + off, pi + off, pd + off, pr ? pr + off : nullptr, HW);
                    }
                    off += 128; row += step_row; col += step_col;
                    if (col >= W) { col -= W; ++row; }
                }
            }
        }
        __syncwarp();      // the key buffer is reused by this warp's next strip
    }
    if (STATS) {
        for (int o = 16; o; o >>= 1) n_tests += __shfl_xor_sync(0xffffffffu, n_tests, o);
        if (lane == 0 && ra.stats) atomicAdd(&ra.stats[0], n_tests);
    }
}

}  // namespace gp
