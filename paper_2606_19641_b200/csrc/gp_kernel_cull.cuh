// gp_kernel_cull.cuh — a1 camera setup + a2 frustum cull and compaction (one warp per view, one CTA per
// group of 8 views of the same world, which share the world's records through shared memory).
//
// For every primitive k != ego of the view's world the kernel
//   1. hoists the (view, primitive) part of contract C5 with the exact contract operations
//      (EntryGeo: a_m, b_m and the camera basis in the box frame);
//   2. decides CONSERVATIVELY, with plain fp32 and explicit error margins, whether the box can
//      touch the view volume (first its bounding sphere, then the box-vs-frustum-plane support
//      test, near / far), and if so bounds its projection by a pixel rectangle (corner
//      projection, edges clipped at the near plane);
//   3. appends survivors to the view's list in global memory (EntryGeo 48 B + EntryAux 16 B).
// Step 2 only ever drops a primitive that cannot produce a contract hit on any pixel centre, and
// the rectangle contains every pixel it can hit, so the rendered planes are bit-identical to the
// all-primitive definition (checked on every pixel against k_render_brute and the CPU oracle).
#pragma once
#include "gp_device.cuh"

namespace gp {

constexpr float kNearEps = 0.01f;      // clip plane for the projection bound, metres of planar depth
constexpr float kNearGuard = 0.05f;    // cross-section this close to the optical centre => whole image

struct PixBounds { float smin, smax, vmin, vmax, xmin; };

// 1/x to ~1 ulp in one MUFU instruction (conservative geometry only; never contract arithmetic)
__device__ __forceinline__ float rcp_fast(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// Projection (s, v) = (Y / X, Z / X) of one camera-frame point with X >= kNearEps, accumulated WITHOUT its error term
// (fast path); bound_widen() then widens the whole interval once by the largest error any accumulated point can have.
__device__ __forceinline__ void bound_point(PixBounds &b, float X, float Y, float Z) {
    const float inv = rcp_fast(X);
    const float s = Y * inv, v = Z * inv;
    b.smin = fminf(b.smin, s); b.smax = fmaxf(b.smax, s);
    b.vmin = fminf(b.vmin, v); b.vmax = fmaxf(b.vmax, v);
    b.xmin = fminf(b.xmin, X);
}
// The same with the point's own error term (precise path: points near the clip plane have large errors that must not
// be charged to the far end of the primitive).  (Y +- E(1+|s|)) / X bounds the true s for an absolute coordinate error
// E; the 1e-6 relative term covers the approximate reciprocal.
__device__ __forceinline__ void bound_point_err(PixBounds &b, float X, float Y, float Z, float E) {
    const float inv = rcp_fast(X);
    const float s = Y * inv, v = Z * inv;
    const float ds = fmaf(E * (1.0f + fabsf(s)), inv, 1e-6f * fabsf(s)), dv = fmaf(E * (1.0f + fabsf(v)), inv, 1e-6f * fabsf(v));
    b.smin = fminf(b.smin, s - ds); b.smax = fmaxf(b.smax, s + ds);
    b.vmin = fminf(b.vmin, v - dv); b.vmax = fmaxf(b.vmax, v + dv);
}
// With |s| <= max|s| and X >= xmin over the accumulated points, the one term below is >= every point's own error term,
// so the widened interval contains each point's own widened interval.  Returns the two widths.
__device__ __forceinline__ void bound_widen(PixBounds &b, float E, float &ds, float &dv) {
    const float inv = rcp_fast(b.xmin) * 1.000001f;
    const float sm = fmaxf(fabsf(b.smin), fabsf(b.smax)), vm = fmaxf(fabsf(b.vmin), fabsf(b.vmax));
    ds = fmaf(E * (1.0f + sm), inv, 1e-6f * sm); dv = fmaf(E * (1.0f + vm), inv, 1e-6f * vm);
    b.smin -= ds; b.smax += ds; b.vmin -= dv; b.vmax += dv;
}

// Does the box (camera frame: centre (Xc, Yc, Zc), half-edge vectors (Xx, Yx, Zx), (Xy, Yy, Zy), (Xz, 0, Zz)) reach
// into the tip cuboid [0, near] x [-gdY, gdY] x [-gdZ, gdZ] of the view pyramid?  Conservative separating-axis test
// over the camera's Y and Z axes (the caller established the overlap in X) and the three box axes.  Out of line: it
// runs only for primitives that straddle the near clip plane, and must not cost the main path registers.
__device__ __noinline__ bool box_meets_tip(float Xc, float Yc, float Zc, float Xx, float Xy, float Xz, float Yx, float Yy,
                                           float Zx, float Zy, float Zz, float near, float gdY, float gdZ, float E) {
    const float Yr = fabsf(Yx) + fabsf(Yy), Zr = fabsf(Zx) + fabsf(Zy) + fabsf(Zz);
    if (!(fabsf(Yc) - Yr < gdY && fabsf(Zc) - Zr < gdZ)) return false;
    const float ex[3] = {Xx, Xy, Xz}, ey[3] = {Yx, Yy, 0.0f}, ez[3] = {Zx, Zy, Zz};   // X, Y, Z parts of the half-edge vectors
#pragma unroll
    for (int m = 0; m < 3; ++m) {
        const float ax = ex[m], ay = ey[m], az = ez[m];
        const float dist = fabsf(ax * (Xc - 0.5f * near) + ay * Yc + az * Zc);
        float r = 0.0f;
#pragma unroll
        for (int q = 0; q < 3; ++q) r += fabsf(ax * ex[q] + ay * ey[q] + az * ez[q]);
        const float rt = fabsf(ax) * (0.5f * near + E) + fabsf(ay) * gdY + fabsf(az) * gdZ;
        if (dist > (r + rt) * 1.0001f + 1e-9f) return false;
    }
    return true;
}

// Camera of the view (contract C2) and everything of C5 that depends only on (view, primitive).
struct CullCam { float ox, oy, oz, fx, fy, rx, ry, ux, uy, cp, sp; };
struct CullPrim {
    EntryGeo g; float olx, oly, olz, hx, hy, hz;
    // conservative camera-frame geometry: centre (Xc, Yc, Zc), half-edge vectors, error bound E
    float E, Xc, Yc, Zc, Xx, Xy, Xz, Yx, Yy, Zx, Zy, Zz, Xr;
};

__device__ __forceinline__ void cull_hoist(const float4 p0 /* cx cy cz hx */, const float4 p1 /* hy hz ck sk */,
                                           const CullCam &c, CullPrim &q) {
    const float pcx = p0.x, pcy = p0.y, pcz = p0.z, ck = p1.z, sk = p1.w;
    q.hx = p0.w; q.hy = p1.x; q.hz = p1.y;
    // ---- contract C5, hoisted part -------------------------------------------------------
    const float ex = c_sub(c.ox, pcx), ey = c_sub(c.oy, pcy);
    q.olx = c_fma(sk, ey, c_mul(ck, ex));
    q.oly = c_fma(ck, ey, -c_mul(sk, ex));
    q.olz = c_sub(c.oz, pcz);
    EntryGeo &g = q.g;
    g.flx = c_fma(sk, c.fy, c_mul(ck, c.fx)); g.fly = c_fma(ck, c.fy, -c_mul(sk, c.fx));
    g.rlx = c_fma(sk, c.ry, c_mul(ck, c.rx)); g.rly = c_fma(ck, c.ry, -c_mul(sk, c.rx));
    g.ulx = c_fma(sk, c.uy, c_mul(ck, c.ux)); g.uly = c_fma(ck, c.uy, -c_mul(sk, c.ux));
    g.ax = c_sub(-q.hx, q.olx); g.bx = c_sub(q.hx, q.olx);
    g.ay = c_sub(-q.hy, q.oly); g.by = c_sub(q.hy, q.oly);
    g.az = c_sub(-q.hz, q.olz); g.bz = c_sub(q.hz, q.olz);
    // ---- conservative geometry (not contract arithmetic) ----------------------------------
    // Camera coordinates of a box-frame point p: X = (p-ol).f_l (planar depth), Y = (p-ol).r_l
    // (right), Z = (p-ol).u_l (up), with f_l = (flx, fly, sp), r_l = (rlx, rly, 0), u_l = (ulx, uly, cp).
    q.E = 1e-5f * (fabsf(q.olx) + fabsf(q.oly) + fabsf(q.olz) + q.hx + q.hy + q.hz) + 1e-6f;
    q.Xc = -(q.olx * g.flx + q.oly * g.fly + q.olz * c.sp);
    q.Yc = -(q.olx * g.rlx + q.oly * g.rly);
    q.Zc = -(q.olx * g.ulx + q.oly * g.uly + q.olz * c.cp);
    q.Xx = q.hx * g.flx; q.Xy = q.hy * g.fly; q.Xz = q.hz * c.sp;        // half-edge vectors, camera frame
    q.Yx = q.hx * g.rlx; q.Yy = q.hy * g.rly;
    q.Zx = q.hx * g.ulx; q.Zy = q.hy * g.uly; q.Zz = q.hz * c.cp;
    q.Xr = fabsf(q.Xx) + fabsf(q.Xy) + fabsf(q.Xz);
}

// Phase-1 test: can the box touch the view volume at all?  (near / far / four side planes, exact
// support function of the box along each plane normal, widened by the error bound.)
__device__ __forceinline__ bool cull_in_frustum(const CullPrim &q, float th, float tv, float t_max) {
    const float E = q.E;
    if (q.Xc + q.Xr < -E) return false;                                   // wholly behind the camera plane
    if (q.Xc - q.Xr > t_max * (1.0f + 1e-6f) + E) return false;           // wholly beyond the far plane
    const float m = E * (2.0f + th + tv);
    float gc, gr;
    gc = q.Yc - th * q.Xc;  gr = fabsf(q.Yx - th * q.Xx) + fabsf(q.Yy - th * q.Xy) + fabsf(th * q.Xz);
    if (gc - gr > m) return false;
    gc = -q.Yc - th * q.Xc; gr = fabsf(q.Yx + th * q.Xx) + fabsf(q.Yy + th * q.Xy) + fabsf(th * q.Xz);
    if (gc - gr > m) return false;
    gc = q.Zc - tv * q.Xc;  gr = fabsf(q.Zx - tv * q.Xx) + fabsf(q.Zy - tv * q.Xy) + fabsf(q.Zz - tv * q.Xz);
    if (gc - gr > m) return false;
    gc = -q.Zc - tv * q.Xc; gr = fabsf(q.Zx + tv * q.Xx) + fabsf(q.Zy + tv * q.Xy) + fabsf(q.Zz + tv * q.Xz);
    if (gc - gr > m) return false;
    return true;
}

// Precise pixel bounds of a box that straddles the clip plane X = near, or has a corner so close to it that the fast path's
// uniform error term is too coarse: corners in front of the plane and the points where edges cross it are projected, each
// with its own error term.  Returns (smin, smax, vmin, vmax); (-inf, inf, -inf, inf) = the whole image.  Out of line: it
// runs for few primitives per view and must not cost the main path registers.
__device__ __noinline__ float4 cull_bounds_precise(float Xc, float Yc, float Zc, float Xx, float Xy, float Xz, float Yx, float Yy,
                                                   float Zx, float Zy, float Zz, float Xr, float E, float th, float tv, bool flat) {
    const float near = kNearEps;
    const float inf = __int_as_float(0x7f800000);
    const float4 whole = make_float4(-inf, inf, -inf, inf);
    if (Xc + Xr < near + E) return whole;                                 // thin sliver in front of the camera plane
    PixBounds b = {3.0e38f, -3.0e38f, 3.0e38f, -3.0e38f, 3.0e38f};
    const int nc = flat ? 4 : 8;                                          // flat: the corners c and c + 4 coincide
    float cX[8], cY[8], cZ[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const float sx = (c & 1) ? 1.0f : -1.0f, sy = (c & 2) ? 1.0f : -1.0f, sz = (c & 4) ? 1.0f : -1.0f;
        cX[c] = Xc + sx * Xx + sy * Xy + sz * Xz;
        cY[c] = Yc + sx * Yx + sy * Yy;
        cZ[c] = Zc + sx * Zx + sy * Zy + sz * Zz;
    }
    float qYmin = 3.0e38f, qYmax = -3.0e38f, qZmin = 3.0e38f, qZmax = -3.0e38f;   // cross-section at X = near
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        if (c >= nc) break;
        if (cX[c] >= near) bound_point_err(b, cX[c], cY[c], cZ[c], E);
#pragma unroll
        for (int bit = 1; bit < 8; bit <<= 1) {
            if ((c & bit) || bit >= nc) continue;
            const int d = c | bit;
            const float Xa = cX[c], Xb = cX[d];
            if ((Xa < near) == (Xb < near)) continue;
            const float t = (near - Xa) * rcp_fast(Xb - Xa);       // |Xb - Xa| > 0 here; error covered by E below
            const float Yi = cY[c] + t * (cY[d] - cY[c]), Zi = cZ[c] + t * (cZ[d] - cZ[c]);
            bound_point_err(b, near, Yi, Zi, E + 1e-6f * (fabsf(cY[d] - cY[c]) + fabsf(cZ[d] - cZ[c])));
            qYmin = fminf(qYmin, Yi); qYmax = fmaxf(qYmax, Yi);
            qZmin = fminf(qZmin, Zi); qZmax = fmaxf(qZmax, Zi);
        }
    }
    // The part of the box with 0 < X < near is not covered by the bound above.  A point of it is inside
    // the image only if |Y| < th X < th near and |Z| < tv near, i.e. only if the box reaches into the tip
    // of the view pyramid; then give up and take the whole image.  Two conservative tests of that: the
    // cross-section at X = near, and the camera-frame bounding intervals of the box, both against the tip
    // widened to at least kNearGuard (the tip is large for extreme fields of view: tv near = 10 m at a
    // 4096 x 4 image).  A box redone here only for precision lies wholly beyond the clip plane: nothing to guard.
    if (Xc - Xr < near + E) {
        const float gdY = fmaxf(kNearGuard, 1.01f * th * near) + E, gdZ = fmaxf(kNearGuard, 1.01f * tv * near) + E;
        if (qYmin <= gdY && qYmax >= -gdY && qZmin <= gdZ && qZmax >= -gdZ) return whole;
        if (fabsf(Yc) - (fabsf(Yx) + fabsf(Yy)) < gdY && fabsf(Zc) - (fabsf(Zx) + fabsf(Zy) + fabsf(Zz)) < gdZ &&
            box_meets_tip(Xc, Yc, Zc, Xx, Xy, Xz, Yx, Yy, Zx, Zy, Zz, near, gdY, gdZ, E))   // rare
            return whole;
    }
    return make_float4(b.smin, b.smax, b.vmin, b.vmax);
}

constexpr int kCullChunk = 320;        // primitives staged in shared memory per round (a multiple of 32)
constexpr int kCullWarps = 8;          // views per CTA (one warp per view), all of the same world

// Launch constants of the cull, formed once on the host (conservative geometry only, no contract arithmetic).
struct CullArgs {
    const gp_prim *prims; const float2 *pitch;
    int world_begin, groups_per_world, H, W;
    float th, tv;
    float sth, stv;                    // |n| of the side planes (-th, +-1, 0) and (-tv, 0, +-1), times 1.0001
    float msc;                         // 2 + th + tv
    float inv_th, inv_tv, halfW, halfH;
    float far_lim;                     // t_max (1 + 1e-6)
    ViewHdr *hdr; EntryGeo *geo; EntryAux *aux; int cap;           // cap: list stride and capacity (entries per view)
    uint8_t *ovf;                      // non-null when cap < P: ovf[view] = 1 if the view's list did not fit
    unsigned long long *stats;
};

// Grid: one CTA per (world, group of kCullWarps views of that world).  The world's records (first 32 bytes of each:
// centre, half extents, heading) are staged in shared memory once per CTA and shared by its views, together with the
// view-independent part of the phase-1 test (bounding-sphere radius with its error margin folded in).
#ifndef GP_CULL_MIN_CTAS
#define GP_CULL_MIN_CTAS 4
#endif
// CAPPED: the lists hold fewer than P entries (GP_OPT_LIST_CAP): overflow is checked and flagged.
template <bool CAPPED>
__global__ void __launch_bounds__(kCullWarps * 32, GP_CULL_MIN_CTAS)
k_cull(SceneConst sc, CullArgs ca) {
    __shared__ float4 s_p0[kCullChunk], s_p1[kCullChunk];
    __shared__ float4 s_c[kCullChunk];                                   // phase 1: centre, R + E_k  (-inf: skip)
    __shared__ float2 s_r[kCullChunk];                                   // phase 1: R sth + E_k msc, R stv + E_k msc
    __shared__ uint8_t s_sphere[kCullChunk];
    __shared__ uint16_t s_idx_all[kCullWarps][kCullChunk];
#if GP_PDL
    // let the render pass (launched with programmatic stream serialisation) start its view-independent prologue as this
    // grid's CTAs drain; it waits (griddepcontrol.wait) for this grid to complete before it reads the lists
    asm volatile("griddepcontrol.launch_dependents;");
#endif
#if GP_PDL
    // ... and this grid may itself have been started early, behind a pose update (k_agents_update / k_dynamics_step): wait
    // for it before the first read of a record (returns at once after a normal launch)
    asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int wl = blockIdx.x / ca.groups_per_world;                    // world within the rendered range
    const int v = (blockIdx.x - wl * ca.groups_per_world) * kCullWarps + warp;   // view within the world
    const int vpw = sc.A * sc.C;
    const bool active = v < vpw;                                        // idle warps still join the barriers
    const int a = sc.C == 1 ? v : v / sc.C, cam_id = v - a * sc.C;
    const int view = wl * vpw + v;
    uint16_t *s_idx = s_idx_all[warp];
    const unsigned lt_mask = (1u << lane) - 1u;
    const int w = ca.world_begin + wl;
    const gp_prim *wp = ca.prims + (size_t)w * sc.P;
    const float th = ca.th, tv = ca.tv;
    const int H = ca.H, W = ca.W;
    CullCam cam = {};
    if (active) {
        const float2 pc = __ldg(&ca.pitch[(size_t)w * sc.A + a]);
        cam.cp = pc.x; cam.sp = pc.y;
        // C2 camera (contract operations)
        const float4 e0 = __ldg(reinterpret_cast<const float4 *>(&wp[a]));        // cx cy cz hx
        const float4 e1 = __ldg(reinterpret_cast<const float4 *>(&wp[a]) + 1);    // hy hz ck sk
        const CamPose cq = rig_camera(sc, cam_id, e0, e1);
        const float e_ck = cq.ck, e_sk = cq.sk;
        cam.ox = cq.ox; cam.oy = cq.oy;
        cam.oz = sc.cam_h;
        cam.fx = c_mul(cam.cp, e_ck); cam.fy = c_mul(cam.cp, e_sk);
        cam.rx = e_sk; cam.ry = -e_ck;
        cam.ux = -c_mul(cam.sp, e_ck); cam.uy = -c_mul(cam.sp, e_sk);
    }

    EntryGeo *vgeo = ca.geo + (size_t)view * ca.cap;
    EntryAux *vaux = ca.aux + (size_t)view * ca.cap;
    int cnt = 0, rmin = 0x1fff;            // list length (warp-uniform), first row touched (per lane)

    // Phase-1 error margin.  The camera-frame coordinates of a centre are formed from d = c - o in fp32; their absolute
    // error is below 1e-5 (|d.x| + |d.y| + |d.z| + R) + 1e-6, and |d.m| <= |c.m| + |o.m|, so the margin splits into a
    // per-primitive part E_k (staged with the record) and a per-view part E_cam.
    const float Ecam = 1.0001e-5f * (fabsf(cam.ox) + fabsf(cam.oy) + fabsf(cam.oz));
    const float EcamM = Ecam * ca.msc;
    const float ninf = __int_as_float(0xff800000);

    for (int k0 = 0; k0 < sc.P; k0 += kCullChunk) {
        const int k1 = min(sc.P, k0 + kCullChunk);
        if (k0) __syncthreads();                                         // previous round fully consumed
        const int npad = (k1 - k0 + 31) & ~31;                           // phase 1 runs whole warps: pad with "skip"
        for (int i = threadIdx.x; i < npad; i += blockDim.x) {
            if (i >= k1 - k0) { s_c[i] = make_float4(0.0f, 0.0f, 0.0f, ninf); s_r[i] = make_float2(0.0f, 0.0f); continue; }
            const float4 *rec = reinterpret_cast<const float4 *>(&wp[k0 + i]);
            float4 p0 = __ldg(rec), p1 = __ldg(rec + 1);
            const bool sphere = __float_as_int(__ldg(rec + 2).z) == GP_SHAPE_SPHERE;     // cls inst shape pad
            if (sphere) { p1.x = p0.w; p1.y = p0.w; p1.z = 1.0f; p1.w = 0.0f; }          // bounding cube, heading 0
            s_p0[i] = p0; s_p1[i] = p1; s_sphere[i] = sphere;
            const float R = sqrtf(fmaf(p0.w, p0.w, fmaf(p1.x, p1.x, p1.y * p1.y))) * 1.0001f;      // bounding-sphere radius
            const float Ek = 1.0001f * fmaf(1e-5f, fabsf(p0.x) + fabsf(p0.y) + fabsf(p0.z) + R, 1e-6f);
            const bool skip = sphere && !sc.spheres;
            s_c[i] = make_float4(p0.x, p0.y, p0.z, skip ? ninf : R + Ek);
            s_r[i] = make_float2(fmaf(R, ca.sth, Ek * ca.msc), fmaf(R, ca.stv, Ek * ca.msc));
        }
        __syncthreads();
        if (!active) continue;
        // ---- phase 1: one primitive per lane: bounding sphere against the view volume in the camera
        // frame (looser than the exact box test of phase 2 by construction: the support of the box
        // along any unit direction is <= R); survivors compacted (ballot) into s_idx
        int m = 0;
#pragma unroll 2
        for (int ib = 0; ib < npad; ib += 32) {
            const int i = ib + lane;
            const float4 c = s_c[i];                                                      // cx cy cz R + E_k
            const float2 r = s_r[i];
            const float dx = c.x - cam.ox, dy = c.y - cam.oy, dz = c.z - cam.oz;
            const float X = fmaf(dx, cam.fx, fmaf(dy, cam.fy, dz * cam.sp));
            const float Y = fmaf(dx, cam.rx, dy * cam.ry);
            const float Z = fmaf(dx, cam.ux, fmaf(dy, cam.uy, dz * cam.cp));
            const float Ra = c.w + Ecam;                                                  // -inf for a skipped record
            // the four slacks (behind the camera plane / beyond the far plane, side planes in Y and in Z), branch-free:
            // pass iff none is negative
            const float t1 = X + Ra, t2 = (ca.far_lim - X) + Ra;
            const float t3 = fmaf(th, X, r.x + EcamM) - fabsf(Y), t4 = fmaf(tv, X, r.y + EcamM) - fabsf(Z);
            const bool pass = fminf(fminf(t1, t2), fminf(t3, t4)) >= 0.0f && k0 + i != a;
            const unsigned mask = __ballot_sync(0xffffffffu, pass);
            if (pass) s_idx[m + __popc(mask & lt_mask)] = (uint16_t)i;
            m += __popc(mask);
        }
        __syncwarp();
        // ---- phase 2: dense over the survivors: exact box-vs-view-volume test, then pixel bounds by
        // corner projection (4 corners for a flat primitive, 8 for a box), list append
        for (int ib = 0; ib < m; ib += 32) {
        const int it = ib + lane;
        bool keep = false;
        EntryGeo g; EntryAux x;
        CullPrim q;
        if (it < m) {
            cull_hoist(s_p0[s_idx[it]], s_p1[s_idx[it]], cam, q);
            keep = cull_in_frustum(q, th, tv, sc.t_max);
        }
        if (keep) {
        const int k = k0 + s_idx[it];
        const bool sphere = s_sphere[s_idx[it]];
        g = q.g;
        if (sphere) {       // C5s entry: e = o - c (ol with heading 0, exact) and r*r; basis slots already world-frame
            g.ax = q.olx; g.bx = q.oly; g.ay = q.olz; g.by = c_mul(q.hx, q.hx);
        }
        const float E = q.E, Xc = q.Xc, Yc = q.Yc, Zc = q.Zc, Xr = q.Xr;
        const float Xx = q.Xx, Xy = q.Xy, Xz = q.Xz, Yx = q.Yx, Yy = q.Yy, Zx = q.Zx, Zy = q.Zy, Zz = q.Zz;
        const bool flat = q.hz == 0.0f;           // flat: the corners c and c + 4 coincide (Xz = Zz = 0)
        PixBounds b = {3.0e38f, -3.0e38f, 3.0e38f, -3.0e38f, 3.0e38f};
        // Fast path: the box lies wholly in front of the clip plane (every corner has X >= near).  Corners are projected
        // without error terms and the rectangle is widened once by the largest error any corner can have; if that costs
        // more than a quarter of a pixel (a corner very close to the camera plane), the precise path redoes it.
        bool precise = !(Xc - Xr >= kNearEps + E);
        if (!precise) {
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const float sx = (c & 1) ? 1.0f : -1.0f, sy = (c & 2) ? 1.0f : -1.0f;
                const float Xb = Xc + sx * Xx + sy * Xy, Yb = Yc + sx * Yx + sy * Yy, Zb = Zc + sx * Zx + sy * Zy;
                bound_point(b, Xb - Xz, Yb, Zb - Zz);
                if (!flat) bound_point(b, Xb + Xz, Yb, Zb + Zz);
            }
            float ds, dv;
            bound_widen(b, E, ds, dv);
            precise = ds * (ca.inv_th * ca.halfW) > 0.25f || dv * (ca.inv_tv * ca.halfH) > 0.25f;
        }
        if (precise) {                                                    // few primitives per view; out of line (registers)
            const float4 pb = cull_bounds_precise(Xc, Yc, Zc, Xx, Xy, Xz, Yx, Yy, Zx, Zy, Zz, Xr, E, th, tv, flat);
            b.smin = pb.x; b.smax = pb.y; b.vmin = pb.z; b.vmax = pb.w;
        }
        // continuous pixel coordinate of s: (s/th + 1) W/2; pixel j is covered iff its centre j + 0.5 is inside
        // (bounds of +-inf, the whole image, clamp to it; an empty accumulation, 3e38 / -3e38, gives c0 > c1)
        const float xl = fminf(fmaxf((b.smin * ca.inv_th + 1.0f) * ca.halfW - 0.52f, -1.0f), (float)W);
        const float xh = fminf(fmaxf((b.smax * ca.inv_th + 1.0f) * ca.halfW - 0.48f, -1.0f), (float)W);
        const float yl = fminf(fmaxf((1.0f - b.vmax * ca.inv_tv) * ca.halfH - 0.52f, -1.0f), (float)H);
        const float yh = fminf(fmaxf((1.0f - b.vmin * ca.inv_tv) * ca.halfH - 0.48f, -1.0f), (float)H);
        const int c0 = max((int)ceilf(xl), 0), c1 = min((int)floorf(xh), W - 1);
        const int r0 = max((int)ceilf(yl), 0), r1 = min((int)floorf(yh), H - 1);
        if (c0 > c1 || r0 > r1) keep = false;                             // touches no pixel centre
        if (keep) rmin = min(rmin, r0);
        x.kf = ((uint32_t)k << 2) | (sphere ? kKindSphere : flat ? kKindFlat : kKindBox);
        x.rows = (uint32_t)r0 | ((uint32_t)r1 << 16);
        x.cols = (uint32_t)c0 | ((uint32_t)c1 << 16);
        x.pad = 0;
        }
        const unsigned kmask = __ballot_sync(0xffffffffu, keep);
        if (keep) {
            const int slot = cnt + __popc(kmask & lt_mask);
            if (!CAPPED || slot < ca.cap) {
                vgeo[slot] = g;
                vaux[slot] = x;
            }
        }
        cnt += __popc(kmask);
        }
        __syncwarp();
    }
    if (!active) return;
    rmin = __reduce_min_sync(0xffffffffu, rmin);
    if (lane == 0) {
        const bool over = CAPPED && cnt > ca.cap; // the list did not fit: draw nothing here, the brute-force repair pass
        if (over) ca.ovf[view] = 1;               // renders this view from the records
        ViewHdr h; h.n = over ? (0x1fff << 19) : (cnt | (rmin << 19)); h.oz = cam.oz; h.cp = cam.cp; h.sp = cam.sp;
        ca.hdr[view] = h;
        if (ca.stats) atomicAdd(&ca.stats[1], (unsigned long long)cnt);
    }
}

}  // namespace gp
