// gp_kernel_cull.cuh — a1 camera setup + a2 frustum cull and compaction (one CTA per view).
//
// For every primitive k != ego of the view's world the kernel
//   1. hoists the (view, primitive) part of contract C5 with the exact contract operations
//      (EntryGeo: a_m, b_m and the camera basis in the box frame);
//   2. decides CONSERVATIVELY, with plain fp32 and explicit error margins, whether the box can
//      touch the view volume (box-vs-frustum-plane support test, near / far), and if so bounds
//      its projection by a pixel rectangle (corner projection, edges clipped at the near plane);
//   3. appends survivors to the view's list in global memory (EntryGeo 48 B + EntryAux 16 B).
// Step 2 only ever drops a primitive that cannot produce a contract hit on any pixel centre, and
// the rectangle contains every pixel it can hit, so the rendered planes are bit-identical to the
// all-primitive definition (checked on every pixel against k_render_brute and the CPU oracle).
#pragma once
#include "gp_device.cuh"

namespace gp {

constexpr float kNearEps = 0.01f;      // clip plane for the projection bound, metres of planar depth
constexpr float kNearGuard = 0.05f;    // cross-section this close to the optical centre => whole image

struct PixBounds { float smin, smax, vmin, vmax; };

__device__ __forceinline__ void bound_point(PixBounds &b, float X, float Y, float Z, float E) {
    // X >= kNearEps.  (Y +- E(1+|s|)) / X bounds the true s for an absolute coordinate error E.
    float inv = 1.0f / X;
    float s = Y * inv, v = Z * inv;
    float ds = E * (1.0f + fabsf(s)) * inv, dv = E * (1.0f + fabsf(v)) * inv;
    b.smin = fminf(b.smin, s - ds); b.smax = fmaxf(b.smax, s + ds);
    b.vmin = fminf(b.vmin, v - dv); b.vmax = fmaxf(b.vmax, v + dv);
}

__global__ void __launch_bounds__(128)
k_cull(SceneConst sc, const gp_prim *__restrict__ prims, const float2 *__restrict__ pitch,
       int world_begin, int H, int W, float th, float tv,
       ViewHdr *__restrict__ hdr, EntryGeo *__restrict__ geo, EntryAux *__restrict__ aux, int cap,
       unsigned long long *__restrict__ stats) {
    __shared__ int s_cnt, s_rmin;
    const int view = blockIdx.x;
    const int w = world_begin + view / sc.A, a = view % sc.A;
    const gp_prim *wp = prims + (size_t)w * sc.P;
    if (threadIdx.x == 0) { s_cnt = 0; s_rmin = 0x1fff; }
    const float2 pc = __ldg(&pitch[(size_t)w * sc.A + a]);
    const float cp = pc.x, sp = pc.y;
    // C2 camera (contract operations)
    const float e_hx = __ldg(&wp[a].hx), e_ck = __ldg(&wp[a].cos_yaw), e_sk = __ldg(&wp[a].sin_yaw);
    const float ox = c_fma(e_hx, e_ck, __ldg(&wp[a].cx)), oy = c_fma(e_hx, e_sk, __ldg(&wp[a].cy));
    const float oz = sc.cam_h;
    const float fx = c_mul(cp, e_ck), fy = c_mul(cp, e_sk);
    const float rx = e_sk, ry = -e_ck;
    const float ux = -c_mul(sp, e_ck), uy = -c_mul(sp, e_sk);
    __syncthreads();

    EntryGeo *vgeo = geo + (size_t)view * cap;
    EntryAux *vaux = aux + (size_t)view * cap;
    const float halfW = 0.5f * (float)W, halfH = 0.5f * (float)H;
    const float inv_th = 1.0f / th, inv_tv = 1.0f / tv;

    for (int k = threadIdx.x; k < sc.P; k += blockDim.x) {
        if (k == a) continue;
        const float4 p0 = __ldg(reinterpret_cast<const float4 *>(&wp[k]));        // cx cy cz hx
        const float4 p1 = __ldg(reinterpret_cast<const float4 *>(&wp[k]) + 1);    // hy hz ck sk
        const float pcx = p0.x, pcy = p0.y, pcz = p0.z, hx = p0.w, hy = p1.x, hz = p1.y, ck = p1.z, sk = p1.w;
        // ---- contract C5, hoisted part -------------------------------------------------------
        const float ex = c_sub(ox, pcx), ey = c_sub(oy, pcy);
        const float olx = c_fma(sk, ey, c_mul(ck, ex));
        const float oly = c_fma(ck, ey, -c_mul(sk, ex));
        const float olz = c_sub(oz, pcz);
        EntryGeo g;
        g.flx = c_fma(sk, fy, c_mul(ck, fx)); g.fly = c_fma(ck, fy, -c_mul(sk, fx));
        g.rlx = c_fma(sk, ry, c_mul(ck, rx)); g.rly = c_fma(ck, ry, -c_mul(sk, rx));
        g.ulx = c_fma(sk, uy, c_mul(ck, ux)); g.uly = c_fma(ck, uy, -c_mul(sk, ux));
        g.ax = c_sub(-hx, olx); g.bx = c_sub(hx, olx);
        g.ay = c_sub(-hy, oly); g.by = c_sub(hy, oly);
        g.az = c_sub(-hz, olz); g.bz = c_sub(hz, olz);

        // ---- conservative geometry (not contract arithmetic) ----------------------------------
        // Camera coordinates of a box-frame point q: X = (q-ol).f_l (planar depth), Y = (q-ol).r_l
        // (right), Z = (q-ol).u_l (up), with f_l = (flx, fly, sp), r_l = (rlx, rly, 0), u_l = (ulx, uly, cp).
        const float E = 1e-5f * (fabsf(olx) + fabsf(oly) + fabsf(olz) + hx + hy + hz) + 1e-6f;
        const float Xc = -(olx * g.flx + oly * g.fly + olz * sp);
        const float Yc = -(olx * g.rlx + oly * g.rly);
        const float Zc = -(olx * g.ulx + oly * g.uly + olz * cp);
        const float Xx = hx * g.flx, Xy = hy * g.fly, Xz = hz * sp;        // half-edge vectors, camera frame
        const float Yx = hx * g.rlx, Yy = hy * g.rly;
        const float Zx = hx * g.ulx, Zy = hy * g.uly, Zz = hz * cp;
        const float Xr = fabsf(Xx) + fabsf(Xy) + fabsf(Xz);
        if (Xc + Xr < -E) continue;                                       // wholly behind the camera plane
        if (Xc - Xr > sc.t_max * (1.0f + 1e-6f) + E) continue;            // wholly beyond the far plane
        {   // support test against the four side planes  +-Y - th X <= 0,  +-Z - tv X <= 0
            const float m = E * (2.0f + th + tv);
            float gc, gr;
            gc = Yc - th * Xc;  gr = fabsf(Yx - th * Xx) + fabsf(Yy - th * Xy) + fabsf(th * Xz);
            if (gc - gr > m) continue;
            gc = -Yc - th * Xc; gr = fabsf(Yx + th * Xx) + fabsf(Yy + th * Xy) + fabsf(th * Xz);
            if (gc - gr > m) continue;
            gc = Zc - tv * Xc;  gr = fabsf(Zx - tv * Xx) + fabsf(Zy - tv * Xy) + fabsf(Zz - tv * Xz);
            if (gc - gr > m) continue;
            gc = -Zc - tv * Xc; gr = fabsf(Zx + tv * Xx) + fabsf(Zy + tv * Xy) + fabsf(Zz + tv * Xz);
            if (gc - gr > m) continue;
        }
        // corner projection with near-plane clipping
        float cX[8], cY[8], cZ[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const float sx = (c & 1) ? 1.0f : -1.0f, sy = (c & 2) ? 1.0f : -1.0f, sz = (c & 4) ? 1.0f : -1.0f;
            cX[c] = Xc + sx * Xx + sy * Xy + sz * Xz;
            cY[c] = Yc + sx * Yx + sy * Yy;
            cZ[c] = Zc + sx * Zx + sy * Zy + sz * Zz;
        }
        PixBounds b = {3.0e38f, -3.0e38f, 3.0e38f, -3.0e38f};
        bool full = false;
        const float near = kNearEps;
        if (Xc - Xr >= near + E) {
#pragma unroll
            for (int c = 0; c < 8; ++c) bound_point(b, cX[c], cY[c], cZ[c], E);
        } else if (Xc + Xr < near + E) {
            full = true;                                                  // thin sliver in front of the camera plane
        } else {
            float qYmin = 3.0e38f, qYmax = -3.0e38f, qZmin = 3.0e38f, qZmax = -3.0e38f;   // cross-section at X = near
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                if (cX[c] >= near) bound_point(b, cX[c], cY[c], cZ[c], E);
#pragma unroll
                for (int bit = 1; bit < 8; bit <<= 1) {
                    if (c & bit) continue;
                    const int d = c | bit;
                    const float Xa = cX[c], Xb = cX[d];
                    if ((Xa < near) == (Xb < near)) continue;
                    const float t = (near - Xa) / (Xb - Xa);
                    const float Yi = cY[c] + t * (cY[d] - cY[c]), Zi = cZ[c] + t * (cZ[d] - cZ[c]);
                    bound_point(b, near, Yi, Zi, E);
                    qYmin = fminf(qYmin, Yi); qYmax = fmaxf(qYmax, Yi);
                    qZmin = fminf(qZmin, Zi); qZmax = fmaxf(qZmax, Zi);
                }
            }
            // the part of the box with 0 < X < near projects outside the bound above only if the
            // cross-section comes close to the optical centre: then give up and take the whole image
            const float gd = kNearGuard + E;
            if (qYmin <= gd && qYmax >= -gd && qZmin <= gd && qZmax >= -gd) full = true;
        }
        int c0, c1, r0, r1;
        if (full) { c0 = 0; c1 = W - 1; r0 = 0; r1 = H - 1; }
        else {
            // continuous pixel coordinate of s: (s/th + 1) W/2; pixel j is covered iff its centre j + 0.5 is inside
            const float xl = fminf(fmaxf((b.smin * inv_th + 1.0f) * halfW - 0.52f, -1.0f), (float)W);
            const float xh = fminf(fmaxf((b.smax * inv_th + 1.0f) * halfW - 0.48f, -1.0f), (float)W);
            const float yl = fminf(fmaxf((1.0f - b.vmax * inv_tv) * halfH - 0.52f, -1.0f), (float)H);
            const float yh = fminf(fmaxf((1.0f - b.vmin * inv_tv) * halfH - 0.48f, -1.0f), (float)H);
            c0 = max((int)ceilf(xl), 0); c1 = min((int)floorf(xh), W - 1);
            r0 = max((int)ceilf(yl), 0); r1 = min((int)floorf(yh), H - 1);
            if (c0 > c1 || r0 > r1) continue;                             // touches no pixel centre
        }
        const int slot = atomicAdd(&s_cnt, 1);
        atomicMin(&s_rmin, r0);
        vgeo[slot] = g;
        EntryAux x;
        x.kf = ((uint32_t)k << 1) | (hz == 0.0f ? 1u : 0u);
        x.rows = (uint32_t)r0 | ((uint32_t)r1 << 16);
        x.cols = (uint32_t)c0 | ((uint32_t)c1 << 16);
        x.pad = 0;
        vaux[slot] = x;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        ViewHdr h; h.n = s_cnt | (s_rmin << 19); h.oz = oz; h.cp = cp; h.sp = sp;
        hdr[view] = h;
        if (stats) atomicAdd(&stats[1], (unsigned long long)s_cnt);
    }
}

}  // namespace gp
