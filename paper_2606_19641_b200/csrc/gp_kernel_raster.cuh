// gp_kernel_raster.cuh — a3-a9, the primitive-major ("rasterisation-style") variant of the render pass
// (PAPER.md:62 "supporting both rasterization and ray tracing", :319 "the rasterizer is faster, exploiting the
// simplicity of the primitives").
//
// The ray path (gp_kernel_render.cuh) is pixel-major: a warp owns a strip of rows and walks the view's list for it,
// so an entry is picked up once per strip it overlaps.  This variant is primitive-major, like a scan-line
// rasteriser with a depth buffer:
//   tile      one CTA owns a tile of TR consecutive rows of one view and a key ("depth") buffer for it in shared memory;
//   scan      the view's list (staged by TMA bulk copy) is taken in chunks of <= 32 entries, chunks handed out to the
//             warps dynamically; a chunk's flat quads are expanded into (entry, row) items, one lane each: the lane
//             bounds the row's column span (the plane depth is fixed per row), finishes short spans itself and hands
//             long ones to the whole warp; boxes / spheres are walked over their pixel rectangle by the whole warp;
//   test      every covered pixel runs the SAME contract test as the ray path (C5 / C5s, exact fp32) and updates the
//             pixel's packed 64-bit key (C6) with an atomic minimum — the depth test of the rasteriser;
//   resolve   after one __syncthreads the warps sweep the tile in groups of 128 pixels: background from the row table,
//             winners patched from the resolve table, the same coalesced stores as the ray path.
// An entry is therefore visited once per tile, not once per strip, and lanes are packed with (entry, row) items that
// really overlap; results are bit-identical to the ray path and to the brute-force kernel by construction (same
// candidate set per pixel, same test, same key order).
#pragma once
#include "gp_kernel_render.cuh"

namespace gp {

#ifndef GP_RASTER_WARPS
#define GP_RASTER_WARPS 4
#endif
#ifndef GP_RASTER_MIN_CTAS
#define GP_RASTER_MIN_CTAS 8
#endif

// Walk of one box / sphere entry over its pixel rectangle clipped to rows [R0, R1], by the whole warp
// (LR rows x LC columns per pass), atomic key updates.
template <bool STATS, bool SPH>
__device__ __forceinline__ unsigned raster_box(const StripBatchCtx &c, const EntryRec &E, int R0, int R1,
                                               unsigned long long *keys, int lane) {
    unsigned n_tests = 0;
    const int W = c.W;
    const float t_max = c.t_max;
    const int LC = 1 << c.log2LC, LR = 32 >> c.log2LC;
    const int li = lane >> c.log2LC, lj = lane & (LC - 1);
    const float4 &g0 = E.g0, &g1 = E.g1, &g2 = E.g2;
    const uint32_t kind = E.ax.x & 3u, klow = (E.ax.x >> 2) << 3;
    const int r0 = max((int)(E.ax.y & 0xffff), R0), r1 = min((int)(E.ax.y >> 16), R1);
    const int c0 = (int)(E.ax.z & 0xffff), c1 = (int)(E.ax.z >> 16);
    for (int rb = r0; rb <= r1; rb += LR) {
        const int i = min(rb + li, r1);                         // lanes past r1 idle (j loop below)
        const bool row_ok = rb + li <= r1;
        const float4 rt = c.s_row[i - R0];                      // v, dz, 1/dz, tg
        unsigned long long *krow = keys + (i - R0) * W;
        if (SPH && kind == kKindSphere) {
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
                        if (key < krow[j]) atomicMin(krow + j, key);
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
                    slab_select<true>(g0, dlx, dly, loz, hiz, rt.y, t_max, false, klow, krow + j);
                }
            }
        }
    }
    return n_tests;
}

// grid: views * ra.ntiles CTAs (tile fastest); block: 2 .. GP_RASTER_WARPS warps.  ra.SR = rows per tile.
template <bool STATS, bool SPH>
__global__ void __launch_bounds__(GP_RASTER_WARPS * 32, GP_RASTER_MIN_CTAS)
k_raster(SceneConst sc, RenderArgs ra) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int H = ra.H, W = ra.W, TR = ra.SR;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, NW = blockDim.x >> 5;
    const int view = blockIdx.x / ra.ntiles, tile = blockIdx.x - view * ra.ntiles;
    const int R0 = tile * TR, R1 = min(H, R0 + TR) - 1, nrows = R1 - R0 + 1;

    // ---- shared memory carve-up ---------------------------------------------------------------
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem);
    int *s_chunk = reinterpret_cast<int *>(smem + 8);              // next chunk of the list to hand out
    uint4 *s_bg = reinterpret_cast<uint4 *>(smem + 16);            // [0] sky, [1] ground: cls4, r4, g4, b4
    EntryGeo *s_geo = reinterpret_cast<EntryGeo *>(smem + 48);
    EntryAux *s_aux = reinterpret_cast<EntryAux *>(smem + 48 + (size_t)ra.scap * 48);
    float4 *s_row = reinterpret_cast<float4 *>(smem + 48 + (size_t)ra.scap * 64);      // [TR]: rows R0 ..
    float *s_col = reinterpret_cast<float *>(s_row + TR);
    unsigned long long *keys = reinterpret_cast<unsigned long long *>(s_col + ((W + 3) & ~3));   // [TR][W]

    const float4 vh4 = __ldg(reinterpret_cast<const float4 *>(&ra.hdr[view]));
    const int hn = __float_as_int(vh4.x);
    const float v_oz = vh4.y, v_cp = vh4.z, v_sp = vh4.w;
    const int n = hn & 0x7ffff, rmin = (int)((uint32_t)hn >> 19);
    const bool busy = n > 0 && R1 >= rmin;                         // else: no entry touches this tile (sky / bare ground)

    if (threadIdx.x == 32 % blockDim.x) {
        const uint32_t g = shade_rgb(sc.pal[1], shade_scale(c_max(sc.Lz, 0.0f), sc.ambient)), k = sc.pal[0];
        s_bg[0] = make_uint4(0u, (k & 0xff) * 0x01010101u, ((k >> 8) & 0xff) * 0x01010101u, ((k >> 16) & 0xff) * 0x01010101u);
        s_bg[1] = make_uint4(0x01010101u, (g & 0xff) * 0x01010101u, ((g >> 8) & 0xff) * 0x01010101u,
                             ((g >> 16) & 0xff) * 0x01010101u);
    }
    if (threadIdx.x == 0 && busy) {
        *s_chunk = 0;
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        const uint32_t ns = (uint32_t)min(n, ra.scap);             // entries beyond scap are read from global memory
        mbar_expect_tx(bar, ns * 64u);
        bulk_g2s(s_geo, ra.geo + (size_t)view * ra.cap, ns * 48u, bar);
        bulk_g2s(s_aux, ra.aux + (size_t)view * ra.cap, ns * 16u, bar);
    }
    // row table of the tile (contract C2-C4), overlapped with the bulk copies
    for (int q = threadIdx.x; q < nrows; q += blockDim.x) {
        const float v = c_mul(c_sub(1.0f, c_mul(c_add((float)(R0 + q), 0.5f), ra.two_over_H)), ra.tv);
        const float dz = c_fma(v, v_cp, v_sp);
        const float inv_z = c_rcp(dz);
        float tg = -1.0f;
        if (dz < 0.0f) {
            const float t = c_mul(c_sub(0.0f, v_oz), inv_z);
            if (t > 0.0f && t <= sc.t_max) tg = t;
        }
        s_row[q] = make_float4(v, dz, inv_z, tg);
    }
    if (busy) {
        for (int j = threadIdx.x; j < W; j += blockDim.x)
            s_col[j] = c_mul(c_sub(c_mul(c_add((float)j, 0.5f), ra.two_over_W), 1.0f), ra.th);
        ulonglong2 *k2 = reinterpret_cast<ulonglong2 *>(keys);
        const int nk2 = nrows * W / 2;                             // nrows * W is a multiple of 4
        for (int q = threadIdx.x; q < nk2; q += blockDim.x) k2[q] = make_ulonglong2(kKeyEmpty, kKeyEmpty);
    }
    __syncthreads();                       // tables, empty keys, mbarrier init visible

    unsigned long long n_tests = 0;
    if (busy) {
        mbar_wait(bar, 0);
        StripBatchCtx sb;
        sb.s_geo = s_geo; sb.g_geo = ra.geo + (size_t)view * ra.cap; sb.s_aux = s_aux; sb.g_aux = ra.aux + (size_t)view * ra.cap;
        sb.s_row = s_row; sb.s_col = s_col; sb.scap = ra.scap; sb.W = W; sb.log2LC = ra.log2LC; sb.th = ra.th; sb.t_max = sc.t_max;
        const float t_max = sc.t_max;
        const int CH = n <= 32 ? 8 : (n <= 96 ? 16 : 32);          // entries per chunk: short lists still feed every warp
        for (;;) {
            int ci = 0;
            if (lane == 0) ci = atomicAdd(s_chunk, 1);
            ci = __shfl_sync(0xffffffffu, ci, 0);
            const int e0 = ci * CH;
            if (e0 >= n) break;
            // ---- a3: lane = entry of the chunk: does it touch the tile's rows? --------------------------------
            const int e = e0 + lane;
            bool ov = false, fl = false;
            int ra0 = 0, cnt = 0;
            if (lane < CH && e < n) {
                const uint2 kr = e < ra.scap ? *reinterpret_cast<const uint2 *>(&s_aux[e])
                                             : __ldg(reinterpret_cast<const uint2 *>(&sb.g_aux[e]));   // kf, rows
                const int er0 = (int)(kr.y & 0xffff), er1 = (int)(kr.y >> 16);
                ov = er0 <= R1 && er1 >= R0;
                fl = (kr.x & 3u) == kKindFlat;
                ra0 = max(er0, R0);
                if (ov && fl) cnt = min(er1, R1) - ra0 + 1;        // (entry, row) items of a flat quad
            }
            const unsigned bmask = __ballot_sync(0xffffffffu, ov && !fl);
            int incl = cnt;                                        // inclusive prefix sum of the item counts
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += y;
            }
            const int total = __shfl_sync(0xffffffffu, incl, 31);
            // ---- flat quads: one lane per (entry, row) item --------------------------------------------------
            for (int t0 = 0; t0 < total; t0 += 32) {
                const int t = t0 + lane;
                int own = 0;                                       // smallest lane whose inclusive count exceeds t
#pragma unroll
                for (int st = 16; st; st >>= 1) {
                    const int y = __shfl_sync(0xffffffffu, incl, own + st - 1);
                    if (y <= t) own += st;
                }
                const int o_incl = __shfl_sync(0xffffffffu, incl, own), o_cnt = __shfl_sync(0xffffffffu, cnt, own);
                const int o_ra = __shfl_sync(0xffffffffu, ra0, own);
                int ja = 1, jb = 0, i = R0, eb = e0;
                if (t < total) {
                    i = o_ra + (t - (o_incl - o_cnt));
                    eb = e0 + own;
                    const EntryRec E = load_entry(sb, eb);
                    const uint32_t klow = (E.ax.x >> 2) << 3;
                    const float4 rt = s_row[i - R0];
                    const int c0 = (int)(E.ax.z & 0xffff), c1 = (int)(E.ax.z >> 16);
                    if (c1 - c0 < kShortSpan) { ja = c0; jb = c1; }    // a few columns only: not worth bounding further
                    else flat_interval(E, rt, sb, ja, jb);
                    if (jb - ja < kShortSpan) {                        // short (or empty): finish it here
                        float loz, hiz;
                        slab_z(E.g1, rt, loz, hiz);
                        unsigned long long *krow = keys + (i - R0) * W;
                        for (int j = ja; j <= jb; ++j) {
                            if (STATS) ++n_tests;
                            const float s = s_col[j];
                            const float dlx = c_fma(rt.x, E.g2.z, c_fma(s, E.g2.x, E.g1.z));
                            const float dly = c_fma(rt.x, E.g2.w, c_fma(s, E.g2.y, E.g1.w));
                            slab_select<true>(E.g0, dlx, dly, loz, hiz, rt.y, t_max, true, klow, krow + j);
                        }
                        jb = ja - 1;                                   // done
                    }
                }
                unsigned lm = __ballot_sync(0xffffffffu, jb >= ja);    // long spans: all lanes, one item at a time
                while (lm) {
                    const int src = __ffs(lm) - 1;
                    lm &= lm - 1;
                    const int bi = __shfl_sync(0xffffffffu, i, src), beb = __shfl_sync(0xffffffffu, eb, src);
                    const int bja = __shfl_sync(0xffffffffu, ja, src), bjb = __shfl_sync(0xffffffffu, jb, src);
                    const EntryRec E = load_entry(sb, beb);
                    const uint32_t bk = (E.ax.x >> 2) << 3;
                    const float4 rt = s_row[bi - R0];
                    float loz, hiz;
                    slab_z(E.g1, rt, loz, hiz);
                    unsigned long long *krow = keys + (bi - R0) * W;
                    for (int j = bja + lane; j <= bjb; j += 32) {
                        if (STATS) ++n_tests;
                        const float s = s_col[j];
                        const float dlx = c_fma(rt.x, E.g2.z, c_fma(s, E.g2.x, E.g1.z));
                        const float dly = c_fma(rt.x, E.g2.w, c_fma(s, E.g2.y, E.g1.w));
                        slab_select<true>(E.g0, dlx, dly, loz, hiz, rt.y, t_max, true, bk, krow + j);
                    }
                }
            }
            // ---- boxes and spheres: the warp walks the entry's pixel rectangle inside the tile -------------------
            unsigned bm = bmask;
            while (bm) {
                const int src = __ffs(bm) - 1;
                bm &= bm - 1;
                const EntryRec E = load_entry(sb, e0 + src);
                n_tests += raster_box<STATS, SPH>(sb, E, R0, R1, keys, lane);
            }
        }
    }
    __syncthreads();                       // every key of the tile is final

    // ---- a5 ground, a7 resolve, a8 shade, a9 store: 128-pixel groups, 4 consecutive pixels per lane ----------
    {
        const int w = ra.world_begin + view / (sc.A * sc.C);
        const uint32_t *wtab = reinterpret_cast<const uint32_t *>(ra.meta + (size_t)w * sc.P);   // uint32[P][8]
        const size_t HW = (size_t)H * W;
        const int npx = nrows * W;
        const size_t o_tile = (size_t)view * HW + (size_t)R0 * W;
        uint8_t *pc0 = ra.o_cls + o_tile;
        int32_t *pi0 = ra.o_inst + o_tile;
        float *pd0 = ra.o_depth + o_tile;
        uint8_t *pr0 = ra.o_rgb ? ra.o_rgb + 2 * (size_t)view * HW + o_tile : nullptr;
        for (int off = warp * 128 + lane * 4; off < npx; off += NW * 128) {
            int row, col;
            if (ra.log2W >= 0) { row = off >> ra.log2W; col = off & (W - 1); }
            else { row = (int)__umulhi((unsigned)off, ra.magicW); col = off - row * W; }
            const unsigned long long *kq = busy ? keys + off : nullptr;
            if (col + 4 <= W)
                resolve_quad(s_row[row].w, s_bg, kq, wtab, pc0 + off, pi0 + off, pd0 + off, pr0 ? pr0 + off : nullptr, HW);
            else
                resolve_quad_split(s_row[row].w, s_row[row + 1].w, W - col, s_bg, kq, wtab, pc0 + off, pi0 + off,
                                   pd0 + off, pr0 ? pr0 + off : nullptr, HW);
        }
    }
    if (STATS) {
        for (int o = 16; o; o >>= 1) n_tests += __shfl_xor_sync(0xffffffffu, n_tests, o);
        if (lane == 0 && ra.stats) atomicAdd(&ra.stats[0], n_tests);
    }
}

}  // namespace gp
