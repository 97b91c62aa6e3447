/* gp_oracle.c — CPU ORACLE for the Gigapixel per-agent perspective render path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It
 * shares no code, header, table or helper with paper_2606_19641_b200/ (the CUDA path)
 * and neither includes the other.
 *
 * What it computes (§3.1 "O_pixel(S_t)": render the state into an
 * ego-centric perspective view; App. A: cuboids for vehicles, planes for
 * road segments, one directional light, per-instance colour; ray tracing per [88],
 * PAPER.md:62/:295).  The paper gives no formula for its renderer, so the plain
 * definition is: for every pixel, cast the ray through the pixel centre and take, over
 * ALL primitives of the world except the ego box, plus the ground plane, the hit with the
 * smallest entry depth.  Three nested plain loops (row, column, primitive); no culling,
 * no lists, no tiles, no SIMD, no threads.
 *
 * Two renderers live here:
 *   orc_render_view  — fp32, following DESIGN.md "Arithmetic contract" C0-C8 operation by
 *                      operation (one rounding per written operation, fmaf only where
 *                      written).  Class/instance ids are an argmin decided by floating
 *                      point, so both sides take that decision in the kernel's precision
 *                      (fp32) along one written expression tree.
 *   orc_shadow_view  — fp64, a DIFFERENT formulation (each box face enumerated as a plane +
 *                      in-rectangle test, world frame, no slabs, no local frame).  It pins
 *                      the fp32 renderer against the contract itself being wrong.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): closed forms CF1-CF6, brute force vs the
 * fp64 face enumeration, invariants I1-I9, the edge rule U10; tests/test_oracle_pitch_pins.py:
 * the pitched camera basis of C2 (f, r, u) on primitives under pitch, from angle-built fp64
 * geometry that does not pass through orc_shadow_view.  Nothing here is
 * "parity unpinned"; none of the pins come from the paper, which prints no value for this
 * path.
 *
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math -mfma -shared -fPIC  (see oracle/build.py)
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

typedef struct {
    float cx, cy, cz;       /* centre, world frame (z up, x forward, y left)          */
    float hx, hy, hz;       /* half extents along the box's own axes, >= 0              */
    float ck, sk;           /* cos / sin of yaw                                         */
    int32_t cls, inst;      /* class id (2 marking, 3 vehicle), user instance id        */
    int32_t shape, pad1;    /* 0 oriented box (flat quad if hz == 0), 1 sphere of radius hx */
} orc_prim;                 /* 48 bytes, the generator's PRIM_DTYPE                      */

typedef struct {
    float cam_height;       /* C2: camera z                                             */
    float t_max;            /* far plane on planar depth, reading U2                    */
    float fov_rad;          /* horizontal field of view                                 */
    float ambient;          /* C8                                                       */
    float light[3];         /* C8, unit vector                                          */
    uint8_t palette[8][3];  /* sky, ground, marking, vehicle, + 4 user classes          */
} orc_params;

/* One camera of the per-agent rig (contract C2, NEXT-2 of SURVEY.md 8(f); "the ego
 * camera is an entity", :319 "number of cameras configurable", :434-435 four cameras: front,
 * front-left, front-right, rear).  cd, sd = cos / sin of the camera's yaw offset from the agent's
 * heading (positive = to the left); mount = position along the agent's x axis in units of its half
 * length (+1 front-centre, 0 centre, -1 rear-centre).  The default (1, 0, 1) is the single front
 * camera of BASELINE.json configs[0]. */
typedef struct { float cd, sd, mount; } orc_cam;

/* C0: min / max that return the non-NaN operand (IEEE minNum / maxNum). */
static float c_min(float a, float b) { if (a != a) return b; if (b != b) return a; return (b < a) ? b : a; }
static float c_max(float a, float b) { if (a != a) return b; if (b != b) return a; return (b > a) ? b : a; }

/* C8: intensity -> 8.8 fixed-point scale -> channel. */
static int shade_scale(float ndl, float ambient)
{
    float diffuse = 1.0f - ambient;
    float I = fmaf(diffuse, ndl, ambient);
    int s8 = (int)(I * 256.0f);
    if (s8 > 256) s8 = 256;
    return s8;
}

/* fp32 contract renderer, one view.  Outputs: cls[H*W] u8, inst[H*W] i32, depth[H*W] f32,
 * rgb[3*H*W] u8 planar (may be NULL), t2[H*W] f32 second-nearest candidate depth (+inf if
 * none; may be NULL), win[H*W] i32 winning primitive index (-1 ground, -2 sky; may be NULL).
 * Returns 0, or -1 on bad arguments. */
int orc_render_view(const orc_prim *prims, int P, int ego, float cp, float sp, const orc_cam *cam,
                    const orc_params *par, int H, int W,
                    uint8_t *cls, int32_t *inst, float *depth, uint8_t *rgb,
                    float *t2_out, int32_t *win_out)
{
    if (!prims || !par || P < 1 || ego < 0 || ego >= P || H < 1 || W < 1) return -1;
    const orc_prim *e = &prims[ego];

    /* C2 camera: mount point on the agent's axis, heading = agent yaw + camera yaw offset */
    float cd = cam ? cam->cd : 1.0f, sd = cam ? cam->sd : 0.0f, mount = cam ? cam->mount : 1.0f;
    float hm = e->hx * mount;
    float ox = fmaf(hm, e->ck, e->cx);
    float oy = fmaf(hm, e->sk, e->cy);
    float oz = par->cam_height;
    float ckc = fmaf(e->ck, cd, -(e->sk * sd));
    float skc = fmaf(e->sk, cd, e->ck * sd);
    float fx = cp * ckc, fy = cp * skc, fz = sp;
    float rx = skc, ry = -ckc, rz = 0.0f;
    float ux = -(sp * ckc), uy = -(sp * skc), uz = cp;
    float th = (float)tan(0.5 * (double)par->fov_rad);
    float tv = th * ((float)H / (float)W);
    float t_max = par->t_max;
    float Lx = par->light[0], Ly = par->light[1], Lz = par->light[2];
    (void)rz; (void)fz; (void)uz;

    for (int i = 0; i < H; ++i) {
        float v = (1.0f - ((float)i + 0.5f) * (2.0f / (float)H)) * tv;
        for (int j = 0; j < W; ++j) {
            float s = (((float)j + 0.5f) * (2.0f / (float)W) - 1.0f) * th;
            /* C3 */
            float dz = fmaf(v, cp, sp);

            float best_t = INFINITY, second_t = INFINITY;
            int best_k = -2;            /* -2 sky, -1 ground, >= 0 primitive */
            int best_m = 2; float best_sigma = 1.0f;

            /* C4 ground */
            if (dz < 0.0f) {
                float tg = (0.0f - oz) * (1.0f / dz);
                if (tg > 0.0f && tg <= t_max) { best_t = tg; best_k = -1; }
            }
            /* C5 every primitive except the ego */
            for (int k = 0; k < P; ++k) {
                if (k == ego) continue;
                const orc_prim *p = &prims[k];
                if (p->shape == 1) {
/* C5s sphere ("traffic lights use spheres"), un-normalised world-frame
                     * direction d, e = o - c.  Foot of the centre on the ray, then the half chord: the
                     * well-conditioned form (no b^2 - ac cancellation). */
                    float dx = fmaf(v, ux, fmaf(s, rx, fx));
                    float dy = fmaf(v, uy, fmaf(s, ry, fy));
                    float ex = ox - p->cx, ey = oy - p->cy, ez = oz - p->cz;
                    float A = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                    float B = fmaf(dz, ez, fmaf(dy, ey, dx * ex));
                    float invA = 1.0f / A;
                    float tca = (-B) * invA;
                    float lx = fmaf(tca, dx, ex), ly = fmaf(tca, dy, ey), lz = fmaf(tca, dz, ez);
                    float l2 = fmaf(lz, lz, fmaf(ly, ly, lx * lx));
                    float h2 = p->hx * p->hx - l2;
                    if (!(h2 >= 0.0f)) continue;
                    float tn = tca - sqrtf(h2 * invA);
                    if (!(tn > 0.0f && tn <= t_max)) continue;
                    int wins = (tn < best_t) || (tn == best_t && best_k < 0);
                    if (wins) { second_t = best_t; best_t = tn; best_k = k; best_m = 3; best_sigma = 1.0f; }
                    else if (tn < second_t) second_t = tn;
                    continue;
                }
                float ck = p->ck, sk = p->sk;
                float ex = ox - p->cx, ey = oy - p->cy;
                float olx = fmaf(sk, ey, ck * ex);
                float oly = fmaf(ck, ey, -(sk * ex));
                float olz = oz - p->cz;
                float flx = fmaf(sk, fy, ck * fx), fly = fmaf(ck, fy, -(sk * fx));
                float rlx = fmaf(sk, ry, ck * rx), rly = fmaf(ck, ry, -(sk * rx));
                float ulx = fmaf(sk, uy, ck * ux), uly = fmaf(ck, uy, -(sk * ux));
                float dlx = fmaf(v, ulx, fmaf(s, rlx, flx));
                float dly = fmaf(v, uly, fmaf(s, rly, fly));
                float dlz = dz;

                float inv, ta, tb;
                inv = 1.0f / dlx; ta = ((-p->hx) - olx) * inv; tb = (p->hx - olx) * inv;
                float lox = c_min(ta, tb), hix = c_max(ta, tb);
                inv = 1.0f / dly; ta = ((-p->hy) - oly) * inv; tb = (p->hy - oly) * inv;
                float loy = c_min(ta, tb), hiy = c_max(ta, tb);
                inv = 1.0f / dlz; ta = ((-p->hz) - olz) * inv; tb = (p->hz - olz) * inv;
                float loz = c_min(ta, tb), hiz = c_max(ta, tb);
                float tn = c_max(c_max(lox, loy), loz);
                float tf = c_min(c_min(hix, hiy), hiz);
                if (!(tn <= tf && tn > 0.0f && tn <= t_max)) continue;

                /* C6: lexicographic (t, k); the ground (k = +inf) loses ties */
                int wins = (tn < best_t) || (tn == best_t && best_k < 0);
                if (wins) {
                    second_t = best_t;
                    best_t = tn; best_k = k;
                    if (p->hz == 0.0f) { best_m = 2; best_sigma = 1.0f; }
                    else {
                        float dm;
                        if (lox == tn) { best_m = 0; dm = dlx; }
                        else if (loy == tn) { best_m = 1; dm = dly; }
                        else { best_m = 2; dm = dlz; }
                        best_sigma = (dm > 0.0f) ? -1.0f : 1.0f;
                    }
                } else if (tn < second_t) {
                    second_t = tn;
                }
            }
            /* the ground was entered first; if a primitive displaced it, it is already in second_t */

            size_t px = (size_t)i * (size_t)W + (size_t)j;
            int c; int32_t id; float dep; int s8 = 256;
            if (best_k == -2) { c = 0; id = -1; dep = 0.0f; }
            else if (best_k == -1) {
                c = 1; id = -1; dep = best_t;
                s8 = shade_scale(c_max(Lz, 0.0f), par->ambient);
            } else {
                const orc_prim *p = &prims[best_k];
                c = p->cls; id = p->inst; dep = best_t;
                float qx = fmaf(p->sk, Ly, p->ck * Lx);
                float qy = fmaf(p->ck, Ly, -(p->sk * Lx));
                float qz = Lz;
                float qm = (best_m == 0) ? qx : (best_m == 1) ? qy : qz;
                s8 = shade_scale(c_max(best_sigma * qm, 0.0f), par->ambient);
                if (best_m == 3) s8 = 256;      /* C8: spheres (lights) are emissive, palette colour unshaded */
            }
            cls[px] = (uint8_t)c; inst[px] = id; depth[px] = dep;
            if (t2_out) t2_out[px] = second_t;
            if (win_out) win_out[px] = best_k;
            if (rgb) {
                size_t plane = (size_t)H * (size_t)W;
                int pc = (c >= 0 && c < 8) ? c : 0;
                for (int ch = 0; ch < 3; ++ch) {
                    int base = par->palette[pc][ch];
                    rgb[(size_t)ch * plane + px] = (uint8_t)((c == 0) ? base : ((base * s8) >> 8));
                }
            }
        }
    }
    return 0;
}

/* fp64 shadow renderer: face enumeration in the world frame.  Outputs win[H*W] (winning
 * primitive index, -1 ground, -2 sky), depth[H*W] (0 for sky), t2[H*W] (second-nearest
 * candidate, +inf if none), ndl[H*W] (max(n.L, 0) of the entry face; 0 for sky). */
int orc_shadow_view(const orc_prim *prims, int P, int ego, float cp_f, float sp_f, const orc_cam *cam,
                    const orc_params *par, int H, int W,
                    int32_t *win, double *depth, double *t2_out, double *ndl_out)
{
    if (!prims || !par || P < 1 || ego < 0 || ego >= P || H < 1 || W < 1) return -1;
    const orc_prim *e = &prims[ego];
    double cp = cp_f, sp = sp_f;
    /* the agent's heading rotated by the camera's yaw offset (2x2 rotation applied to the unit
     * heading vector), mount point along the agent's own axis */
    double cd = cam ? cam->cd : 1.0, sd = cam ? cam->sd : 0.0, mount = cam ? cam->mount : 1.0;
    double ack = e->ck, ask = e->sk;
    double o[3] = { (double)e->cx + mount * (double)e->hx * ack, (double)e->cy + mount * (double)e->hx * ask,
                    (double)par->cam_height };
    double eck = cd * ack - sd * ask, esk = sd * ack + cd * ask;
    double f[3] = { cp * eck, cp * esk, sp };
    double r[3] = { esk, -eck, 0.0 };
    double u[3] = { -sp * eck, -sp * esk, cp };
    double th = (double)(float)tan(0.5 * (double)par->fov_rad);
    double tv = th * (double)H / (double)W;
    double t_max = par->t_max;
    double L[3] = { par->light[0], par->light[1], par->light[2] };

    for (int i = 0; i < H; ++i) {
        double v = (1.0 - (i + 0.5) * 2.0 / H) * tv;
        for (int j = 0; j < W; ++j) {
            double s = ((j + 0.5) * 2.0 / W - 1.0) * th;
            double d[3];
            for (int a = 0; a < 3; ++a) d[a] = f[a] + s * r[a] + v * u[a];

            double best_t = INFINITY, second_t = INFINITY, best_ndl = 0.0;
            int best_k = -2;
            if (d[2] < 0.0) {
                double tg = -o[2] / d[2];
                if (tg > 0.0 && tg <= t_max) {
                    best_t = tg; best_k = -1; best_ndl = L[2] > 0.0 ? L[2] : 0.0;
                }
            }
            for (int k = 0; k < P; ++k) {
                if (k == ego) continue;
                const orc_prim *p = &prims[k];
                if (p->shape == 1) {
/* quadratic |e + t d|^2 = r^2 solved directly (fp64 affords the cancellation) */
                    double e3[3] = { o[0] - p->cx, o[1] - p->cy, o[2] - p->cz };
                    double qa = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
                    double qb = e3[0] * d[0] + e3[1] * d[1] + e3[2] * d[2];
                    double qc = e3[0] * e3[0] + e3[1] * e3[1] + e3[2] * e3[2] - (double)p->hx * (double)p->hx;
                    double disc = qb * qb - qa * qc;
                    if (disc < 0.0) continue;
                    double ts = (-qb - sqrt(disc)) / qa;
                    if (!(ts > 0.0 && ts <= t_max)) continue;
                    int winss = (ts < best_t) || (ts == best_t && best_k < 0);
                    if (winss) { second_t = best_t; best_t = ts; best_k = k; best_ndl = 1.0; }
                    else if (ts < second_t) second_t = ts;
                    continue;
                }
                double c[3] = { p->cx, p->cy, p->cz };
                double h[3] = { p->hx, p->hy, p->hz };
                double ax[3][3] = { { p->ck, p->sk, 0.0 }, { -(double)p->sk, p->ck, 0.0 }, { 0.0, 0.0, 1.0 } };
                int flat = (p->hz == 0.0f);
                double hit_t = INFINITY, hit_ndl = 0.0;
                for (int m = 0; m < 3; ++m) {
                    if (flat && m != 2) continue;
                    for (int sg = -1; sg <= 1; sg += 2) {
                        double n[3] = { sg * ax[m][0], sg * ax[m][1], sg * ax[m][2] };
                        double denom = n[0] * d[0] + n[1] * d[1] + n[2] * d[2];
                        if (flat) { if (denom == 0.0) continue; }
                        else if (!(denom < 0.0)) continue;          /* entry faces face the ray */
                        double fc[3] = { c[0] + sg * h[m] * ax[m][0], c[1] + sg * h[m] * ax[m][1],
                                         c[2] + sg * h[m] * ax[m][2] };
                        double num = n[0] * (fc[0] - o[0]) + n[1] * (fc[1] - o[1]) + n[2] * (fc[2] - o[2]);
                        double t = num / denom;
                        if (!(t > 0.0 && t <= t_max)) continue;
                        double q[3] = { o[0] + t * d[0] - c[0], o[1] + t * d[1] - c[1], o[2] + t * d[2] - c[2] };
                        int inside = 1;
                        for (int mm = 0; mm < 3; ++mm) {
                            if (mm == m) continue;
                            double a = q[0] * ax[mm][0] + q[1] * ax[mm][1] + q[2] * ax[mm][2];
                            if (fabs(a) > h[mm]) inside = 0;
                        }
                        if (!inside) continue;
                        if (t < hit_t) {
                            hit_t = t;
                            /* flat primitives are shaded with the upward normal (C8) */
                            double nl = flat ? L[2] : (n[0] * L[0] + n[1] * L[1] + n[2] * L[2]);
                            hit_ndl = nl > 0.0 ? nl : 0.0;
                        }
                        if (flat) break;                              /* one plane, either side */
                    }
                }
                if (hit_t == INFINITY) continue;
                int wins = (hit_t < best_t) || (hit_t == best_t && best_k < 0);
                if (wins) { second_t = best_t; best_t = hit_t; best_k = k; best_ndl = hit_ndl; }
                else if (hit_t < second_t) second_t = hit_t;
            }
            size_t px = (size_t)i * (size_t)W + (size_t)j;
            win[px] = best_k;
            depth[px] = (best_k == -2) ? 0.0 : best_t;
            if (t2_out) t2_out[px] = second_t;
            if (ndl_out) ndl_out[px] = (best_k == -2) ? 0.0 : best_ndl;
        }
    }
    return 0;
}

/* C1p: polyline -> thin planar strips (PAPER.md:62 "lane polylines ... thin planar strips", :331 "road
 * geometry, encoded as polyline segments").  pts: [n_lines][pts_per_line][2] fp32 (x, y).  Segment s of
 * line l becomes flat quad number q = l * (pts_per_line - 1) + s: centre at the segment's midpoint,
 * half length along the segment, heading = the normalised segment direction (heading (1, 0) for a
 * zero-length segment), half width / height / class as given, inst = inst0 + q.  fp32, one rounding
 * per written operation (C1p).  Returns the number of quads written. */
int orc_polyline_quads(const float *pts, int n_lines, int pts_per_line, float half_width, float z,
                       int cls, int inst0, orc_prim *out)
{
    if (!pts || !out || n_lines < 0 || pts_per_line < 2) return -1;
    int q = 0;
    for (int l = 0; l < n_lines; ++l) {
        for (int s = 0; s + 1 < pts_per_line; ++s, ++q) {
            const float *p0 = pts + ((size_t)l * pts_per_line + s) * 2, *p1 = p0 + 2;
            float dx = p1[0] - p0[0], dy = p1[1] - p0[1];
            float len = sqrtf(fmaf(dy, dy, dx * dx));
            float ck = 1.0f, sk = 0.0f;
            if (len > 0.0f) { float inv = 1.0f / len; ck = dx * inv; sk = dy * inv; }
            orc_prim *o = &out[q];
            o->cx = fmaf(0.5f, dx, p0[0]); o->cy = fmaf(0.5f, dy, p0[1]); o->cz = z;
            o->hx = 0.5f * len; o->hy = half_width; o->hz = 0.0f;
            o->ck = ck; o->sk = sk;
            o->cls = cls; o->inst = inst0 + q; o->shape = 0; o->pad1 = 0;
        }
    }
    return q;
}
