// gp_kernels_basic.cuh — a0 (pose update, shading table) and the brute-force reference kernel.
#pragma once
#include "gp_device.cuh"

namespace gp {

// C8 hoisted per primitive: the six face intensities.  One thread per primitive of worlds
// [0, Wn) restricted to k < k_end (k_end = A refreshes only the agents).
__device__ __forceinline__ void write_meta(const gp_prim &p, PrimMeta *out, const SceneConst &sc) {
    float qx = c_fma(p.sin_yaw, sc.Ly, c_mul(p.cos_yaw, sc.Lx));
    float qy = c_fma(p.cos_yaw, sc.Ly, -c_mul(p.sin_yaw, sc.Lx));
    float q[3] = {qx, qy, sc.Lz};
    PrimMeta m;
    m.inst = p.inst; m.inst_dup = p.inst;
    const uint32_t c = (uint32_t)p.cls & 7u;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const int lo = shade_scale(c_max(-q[a], 0.0f), sc.ambient);    // sigma = -1
        const int hi = shade_scale(c_max(q[a], 0.0f), sc.ambient);     // sigma = +1
        const bool plain = c == 0 || p.shape == GP_SHAPE_SPHERE;       // sky colour / emissive sphere: unshaded
        m.face[a * 2 + 0] = (plain ? sc.pal[c] : shade_rgb(sc.pal[c], lo)) | (c << 24);
        m.face[a * 2 + 1] = (plain ? sc.pal[c] : shade_rgb(sc.pal[c], hi)) | (c << 24);
    }
    *out = m;
}

__global__ void k_prim_meta(SceneConst sc, const gp_prim *__restrict__ prims, PrimMeta *__restrict__ meta) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    size_t n = (size_t)sc.Wn * sc.P;
    if (i >= n) return;
    write_meta(prims[i], &meta[i], sc);
}

// a0: pose[Wn][A][4] = (cx, cy, cos, sin) -> agent records + their shading table.
__global__ void k_agents_update(SceneConst sc, const float4 *__restrict__ pose, gp_prim *__restrict__ prims,
                                PrimMeta *__restrict__ meta) {
    // a cull launched behind this kernel with programmatic stream serialisation may become resident now (it waits for
    // this grid to complete before it reads a record)
#if GP_PDL
    asm volatile("griddepcontrol.launch_dependents;");
#endif
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    size_t n = (size_t)sc.Wn * sc.A;
    if (i >= n) return;
    size_t w = i / sc.A, a = i % sc.A;
    float4 ps = __ldg(&pose[i]);
    gp_prim *p = &prims[w * sc.P + a];
    p->cx = ps.x; p->cy = ps.y; p->cos_yaw = ps.z; p->sin_yaw = ps.w;
    gp_prim q = *p;
    write_meta(q, &meta[w * sc.P + a], sc);
}

// a0 for static slots: records copied from device memory + their shading table.
__global__ void k_statics_update(SceneConst sc, const gp_prim *__restrict__ src, int n, int q_begin,
                                 gp_prim *__restrict__ prims, PrimMeta *__restrict__ meta) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (size_t)sc.Wn * n) return;
    const size_t w = i / n, q = i % n;
    const gp_prim p = src[i];
    const size_t k = w * sc.P + sc.A + q_begin + q;
    prims[k] = p;
    write_meta(p, &meta[k], sc);
}

// C1p: one thread per polyline segment -> flat quad record + its shading table.
__global__ void k_polyline_quads(SceneConst sc, const float2 *__restrict__ pts, int n_lines, int pts_per_line,
                                 float half_width, float z, int cls, int q_begin, gp_prim *__restrict__ prims,
                                 PrimMeta *__restrict__ meta) {
    const int segs = pts_per_line - 1, per_world = n_lines * segs;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (size_t)sc.Wn * per_world) return;
    const int w = (int)(i / per_world), q = (int)(i % per_world);
    const int l = q / segs, s = q - l * segs;
    const float2 *p = pts + ((size_t)w * n_lines + l) * pts_per_line + s;
    const float2 p0 = __ldg(p), p1 = __ldg(p + 1);
    const float dx = c_sub(p1.x, p0.x), dy = c_sub(p1.y, p0.y);
    const float len = c_sqrt(c_fma(dy, dy, c_mul(dx, dx)));
    float ck = 1.0f, sk = 0.0f;
    if (len > 0.0f) { const float inv = c_rcp(len); ck = c_mul(dx, inv); sk = c_mul(dy, inv); }
    gp_prim o;
    o.cx = c_fma(0.5f, dx, p0.x); o.cy = c_fma(0.5f, dy, p0.y); o.cz = z;
    o.hx = c_mul(0.5f, len); o.hy = half_width; o.hz = 0.0f;
    o.cos_yaw = ck; o.sin_yaw = sk;
    o.cls = cls; o.inst = sc.A + q_begin + q; o.shape = GP_SHAPE_BOX; o.pad = 0;
    const size_t k = (size_t)w * sc.P + sc.A + q_begin + q;
    prims[k] = o;
    write_meta(o, &meta[k], sc);
}

__global__ void k_fill_pitch(float2 *pitch, size_t n) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) pitch[i] = make_float2(1.0f, 0.0f);
}

// Brute force (GP_PATH_BRUTE): one thread per pixel, every primitive of the world straight from the
// 48-byte records, contract C2-C8 with nothing hoisted, scalar stores.  Any H, W.  It is the
// on-device cross-check of the fast path (tests compare the two on every pixel) and is itself
// compared with the CPU oracle.
__global__ void __launch_bounds__(256)
k_render_brute(SceneConst sc, const gp_prim *__restrict__ prims, const float2 *__restrict__ pitch,
               int world_begin, int H, int W, float th, float tv,
               uint8_t *__restrict__ o_cls, int32_t *__restrict__ o_inst, float *__restrict__ o_depth,
               uint8_t *__restrict__ o_rgb, const uint8_t *__restrict__ only_flagged) {
    const int view = blockIdx.x;
    if (only_flagged && !only_flagged[view]) return;    // repair pass of a capped list (GP_OPT_LIST_CAP): flagged views only
    const int va = view / sc.C, cam = view - va * sc.C;
    const int w = world_begin + va / sc.A, a = va % sc.A;
    const gp_prim *wp = prims + (size_t)w * sc.P;
    const float2 pc = pitch[(size_t)w * sc.A + a];
    const float cp = pc.x, sp = pc.y;
    const gp_prim e = wp[a];
    // C2
    const CamPose cq = rig_camera(sc, cam, make_float4(e.cx, e.cy, e.cz, e.hx), make_float4(e.hy, e.hz, e.cos_yaw, e.sin_yaw));
    const float ox = cq.ox, oy = cq.oy, oz = sc.cam_h;
    const float fx = c_mul(cp, cq.ck), fy = c_mul(cp, cq.sk);
    const float rx = cq.sk, ry = -cq.ck;
    const float ux = -c_mul(sp, cq.ck), uy = -c_mul(sp, cq.sk);
    const int HW = H * W;
    for (int px = blockIdx.y * blockDim.x + threadIdx.x; px < HW; px += gridDim.y * blockDim.x) {
        const int i = px / W, j = px - i * W;
        const float s = pix_s(j, W, th), v = pix_v(i, H, tv);
        const float dz = c_fma(v, cp, sp);
        const float inv_z = c_rcp(dz);
        float best_t = __int_as_float(0x7f800000);
        int best_k = -2, best_m = 2; float best_sigma = 1.0f;
        if (dz < 0.0f) {
            float tg = c_mul(c_sub(0.0f, oz), inv_z);
            if (tg > 0.0f && tg <= sc.t_max) { best_t = tg; best_k = -1; }
        }
        for (int k = 0; k < sc.P; ++k) {
            if (k == a) continue;
            const gp_prim p = wp[k];
            if (p.shape == GP_SHAPE_SPHERE) {                       // C5s
                if (!sc.spheres) continue;
                const float dx = c_fma(v, ux, c_fma(s, rx, fx)), dy = c_fma(v, uy, c_fma(s, ry, fy));
                const float tn = sphere_entry(c_sub(ox, p.cx), c_sub(oy, p.cy), c_sub(oz, p.cz), c_mul(p.hx, p.hx), dx, dy, dz);
                if (!(tn > 0.0f && tn <= sc.t_max)) continue;
                if (tn < best_t || (tn == best_t && best_k < 0)) { best_t = tn; best_k = k; best_m = 3; best_sigma = 1.0f; }
                continue;
            }
            const float ck = p.cos_yaw, sk = p.sin_yaw;
            const float ex = c_sub(ox, p.cx), ey = c_sub(oy, p.cy);
            const float olx = c_fma(sk, ey, c_mul(ck, ex));
            const float oly = c_fma(ck, ey, -c_mul(sk, ex));
            const float olz = c_sub(oz, p.cz);
            const float flx = c_fma(sk, fy, c_mul(ck, fx)), fly = c_fma(ck, fy, -c_mul(sk, fx));
            const float rlx = c_fma(sk, ry, c_mul(ck, rx)), rly = c_fma(ck, ry, -c_mul(sk, rx));
            const float ulx = c_fma(sk, uy, c_mul(ck, ux)), uly = c_fma(ck, uy, -c_mul(sk, ux));
            const float dlx = c_fma(v, ulx, c_fma(s, rlx, flx));
            const float dly = c_fma(v, uly, c_fma(s, rly, fly));
            float inv, ta, tb;
            inv = c_rcp(dlx); ta = c_mul(c_sub(-p.hx, olx), inv); tb = c_mul(c_sub(p.hx, olx), inv);
            const float lox = c_min(ta, tb), hix = c_max(ta, tb);
            inv = c_rcp(dly); ta = c_mul(c_sub(-p.hy, oly), inv); tb = c_mul(c_sub(p.hy, oly), inv);
            const float loy = c_min(ta, tb), hiy = c_max(ta, tb);
            ta = c_mul(c_sub(-p.hz, olz), inv_z); tb = c_mul(c_sub(p.hz, olz), inv_z);
            const float loz = c_min(ta, tb), hiz = c_max(ta, tb);
            const float tn = c_max(c_max(lox, loy), loz);
            const float tf = c_min(c_min(hix, hiy), hiz);
            if (!(tn <= tf && tn > 0.0f && tn <= sc.t_max)) continue;
            if (tn < best_t || (tn == best_t && best_k < 0)) {       // C6: ascending k, ground loses ties
                best_t = tn; best_k = k;
                if (p.hz == 0.0f) { best_m = 2; best_sigma = 1.0f; }
                else {
                    float dm;
                    if (lox == tn) { best_m = 0; dm = dlx; }
                    else if (loy == tn) { best_m = 1; dm = dly; }
                    else { best_m = 2; dm = dz; }
                    best_sigma = dm > 0.0f ? -1.0f : 1.0f;
                }
            }
        }
        int c, id, s8 = 256; float dep;
        if (best_k == -2) { c = 0; id = -1; dep = 0.0f; }
        else if (best_k == -1) { c = 1; id = -1; dep = best_t; s8 = shade_scale(c_max(sc.Lz, 0.0f), sc.ambient); }
        else {
            const gp_prim p = wp[best_k];
            c = p.cls & 7; id = p.inst; dep = best_t;             // unvalidated device records: same mask as the resolve table
            const float qx = c_fma(p.sin_yaw, sc.Ly, c_mul(p.cos_yaw, sc.Lx));
            const float qy = c_fma(p.cos_yaw, sc.Ly, -c_mul(p.sin_yaw, sc.Lx));
            const float qm = best_m == 0 ? qx : best_m == 1 ? qy : sc.Lz;
            s8 = shade_scale(c_max(c_mul(best_sigma, qm), 0.0f), sc.ambient);
            if (best_m == 3) s8 = 256;                              // C8: spheres are emissive
        }
        const size_t o = (size_t)view * HW + px;
        o_cls[o] = (uint8_t)c; o_inst[o] = id; o_depth[o] = dep;
        if (o_rgb) {
            const uint32_t pal = sc.pal[c & 7];
            const uint32_t rgb = c == 0 ? pal : shade_rgb(pal, s8);
            const size_t ob = (size_t)view * 3 * HW + px;
            o_rgb[ob] = (uint8_t)(rgb & 0xff); o_rgb[ob + HW] = (uint8_t)((rgb >> 8) & 0xff);
            o_rgb[ob + 2 * (size_t)HW] = (uint8_t)((rgb >> 16) & 0xff);
        }
    }
}

}  // namespace gp
