/* gp_sim_oracle.c — CPU ORACLE for the step either side of the render:
 * the jerk-actuated kinematic bicycle and the vectorised observation O_vec.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.  It shares no code, header, table or
 * helper with paper_2606_19641_b200/ (the CUDA path) and neither includes the other.
 *
 * orc_dynamics_step — PAPER.md:335: "Each agent is controlled through a discrete set of twelve actions, formed
 *   as the Cartesian product of longitudinal jerk values {-15, -4, 0, 4} m/s^3 and lateral jerk values {-4, 0, 4}
 *   m/s^3, which drive a jerk-actuated kinematic bicycle model.  At each step the selected jerks are integrated
 *   into longitudinal and lateral accelerations and then into velocity and steering, with accelerations clipped to
 *   g-force limits, speed clipped to the speed limit, and the steering angle and its rate bounded [...].  The
 *   wheelbase is set to 60% of the vehicle length."  The paper defers the derivation to another paper, so the
 *   order of operations is the reading D1-D6 of DESIGN.md "Dynamics contract", followed here step by step in
 *   fp64 (inputs are the fp32 arrays the kernel consumes, outputs are rounded to fp32 once at the end).  The
 *   path contains atan / tan / cos / sin, so parity with the fp32 kernel is by tolerance (DESIGN.md derives it).
 *
 * orc_observe_vec — PAPER.md:331: "surrounding agents (the nearest K within 100 m), each contributing relative
 *   position, dimensions, relative heading as (cos, sin), and relative signed speed; road geometry, encoded as
 *   polyline segments retrieved from a spatial hash around the agent, each carrying relative position, length,
 *   orientation as (cos, sin), and a categorical type".  The plain definition: for every agent, ALL other agents
 *   (all road segments) of its world are examined, those within the radius are ordered by (squared distance,
 *   index) and the first K (M) are reported.  No spatial hash: that is an acceleration structure, it changes
 *   nothing in the result.  Which neighbours are nearest is an integer decision taken by floating point, so
 *   the squared distance is formed in fp32 along one written expression (contract O1 of DESIGN.md), and so are
 *   the reported features (O2-O3: only fp32 add / mul / fma, no transcendental); parity is bit-exact.
 *
 * Pins (tests/test_oracle_sim_pins.py, -m "not gpu"): closed forms of straight-line motion under constant
 * jerk, the constant-curvature arc, saturation at every limit, the action table; for O_vec hand-placed
 * neighbours (ahead / left / behind, heading differences), the radius boundary, tie order, padding, and an
 * independent fp64 argsort on tie-free random scenes.  Nothing here is "parity unpinned"; the paper prints
 * no value for either operation.
 *
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math -mfma -shared -fPIC  (oracle/build.py)
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

/* ---------------------------------------------------------------------------------------------- dynamics */

typedef struct {
    float dt;               /* step, s (0.1)                                                          */
    float a_lon_max;        /* |longitudinal acceleration| limit, m/s^2 ("g-force limits")            */
    float a_lat_max;        /* |lateral acceleration| limit, m/s^2                                    */
    float v_max;            /* speed limit, m/s; speed is clipped to [0, v_max] (no reversing)        */
    float steer_max;        /* |steering angle| limit, rad                                            */
    float steer_rate_max;   /* |steering rate| limit, rad/s                                           */
    float v_eps;            /* speed below which the curvature demand uses v_eps (avoids 1/0), m/s    */
    float extent;           /* > 0: positions wrap onto the torus [-extent/2, extent/2) (reading U15) */
} orc_dyn_params;

static const double JLON[4] = { -15.0, -4.0, 0.0, 4.0 };
static const double JLAT[3] = { -4.0, 0.0, 4.0 };

static double clipd(double x, double lo, double hi) { return x < lo ? lo : (x > hi ? hi : x); }

/* One step for n agents.  action[n] in [0, 12): longitudinal jerk index = action / 3, lateral = action % 3.
 * state[n][8] fp32 in/out: v, a_lon, a_lat, steer, psi, 3 unused.  pose[n][4] fp32 in/out: x, y, cos psi, sin psi
 * (the buffer the renderer's pose update consumes).  half_len[n]: half length hx of each agent's box (wheelbase =
 * 0.6 * 2 hx).  Returns 0, or -1 on bad arguments (an action outside [0, 12) or a half length <= 0 leaves that agent
 * untouched and makes the call return -2 after processing the others). */
int orc_dynamics_step(const orc_dyn_params *par, int n, const int32_t *action, const float *half_len,
                      float *state, float *pose)
{
    if (!par || !action || !half_len || !state || !pose || n < 0) return -1;
    int rc = 0;
    const double dt = par->dt;
    for (int i = 0; i < n; ++i) {
        int a = action[i];
        if (a < 0 || a >= 12) { rc = -2; continue; }
        if (!(half_len[i] > 0.0f)) { rc = -2; continue; }     /* no length, no wheelbase: untouched, like an invalid action */
        float *s = state + (size_t)i * 8, *p = pose + (size_t)i * 4;
        double v = s[0], a_lon = s[1], a_lat = s[2], steer = s[3], psi = s[4];
        double x = p[0], y = p[1];
        /* D1: jerks -> accelerations, clipped to the g-force limits */
        a_lon = clipd(a_lon + JLON[a / 3] * dt, -(double)par->a_lon_max, par->a_lon_max);
        a_lat = clipd(a_lat + JLAT[a % 3] * dt, -(double)par->a_lat_max, par->a_lat_max);
        /* D2: longitudinal acceleration -> speed, clipped to [0, speed limit] */
        v = clipd(v + a_lon * dt, 0.0, par->v_max);
        /* D3: lateral acceleration -> steering.  a_lat = v^2 kappa and kappa = tan(steer) / L for the kinematic
         * bicycle with wheelbase L = 0.6 * length; the demanded angle is bounded in rate, then in magnitude */
        double L = 0.6 * (2.0 * (double)half_len[i]);
        double vv = v > (double)par->v_eps ? v : (double)par->v_eps;
        double want = atan(L * a_lat / (vv * vv));
        double dmax = (double)par->steer_rate_max * dt;
        steer = steer + clipd(want - steer, -dmax, dmax);
        steer = clipd(steer, -(double)par->steer_max, par->steer_max);
        /* D4: heading, wrapped into [-pi, pi) */
        psi = psi + v * (tan(steer) / L) * dt;
        const double PI = 3.14159265358979323846;
        if (fabs(psi) > 2.0 * PI) psi = remainder(psi, 2.0 * PI);     /* more than a full turn in one step */
        if (psi >= PI) psi -= 2.0 * PI;
        if (psi < -PI) psi += 2.0 * PI;
        /* D5: position with the NEW speed and heading (semi-implicit Euler) */
        double c = cos(psi), sn = sin(psi);
        x = x + v * c * dt;
        y = y + v * sn * dt;
        /* D6: torus wrap of the position (optional) */
        if (par->extent > 0.0f) {
            double E = par->extent, h = 0.5 * E;
            if (x >= h) x -= E;
            if (x < -h) x += E;
            if (y >= h) y -= E;
            if (y < -h) y += E;
        }
        s[0] = (float)v; s[1] = (float)a_lon; s[2] = (float)a_lat; s[3] = (float)steer; s[4] = (float)psi;
        p[0] = (float)x; p[1] = (float)y; p[2] = (float)c; p[3] = (float)sn;
    }
    return rc;
}

/* ------------------------------------------------------------------------------------- vectorised observation */

typedef struct {            /* the renderer's 48-byte primitive record (generator PRIM_DTYPE) */
    float cx, cy, cz, hx, hy, hz, ck, sk;
    int32_t cls, inst, shape, pad1;
} orc_prim48;

/* O_vec of one world.  prims[P]: agents 0..A-1 then statics.  speed[A]: signed longitudinal speed of each agent.
 * For every agent i (ego frame: origin at its box centre, x along its heading, y to its left):
 *   agent_idx[A][K]  int32: indices j != i of the K nearest agents with d2 <= radius^2, ascending (d2, j); -1 pads
 *   agent_feat[A][K][8] fp32: rel x, rel y, length, width, cos(psi_j - psi_i), sin(psi_j - psi_i), v_j - v_i, 1; zeros pad
 *   road_idx[A][M]   int32: primitive indices k >= A of the M nearest road segments (statics with hz == 0 that are
 *                    not spheres), by their centre, with d2 <= radius^2, ascending (d2, k); -1 pads
 *   road_feat[A][M][8] fp32: rel x, rel y of the centre, length, cos / sin of the segment's direction in the ego
 *                    frame, type (= cls as a float), 1, 0; zeros pad
 * Contract (fp32, one rounding per written operation, fmaf only where written):
 *   O1  dx = x_j - x_i; dy = y_j - y_i; d2 = fmaf(dy, dy, dx * dx); within iff d2 <= radius * radius
 *   O2  rel x = fmaf(s_i, dy, c_i * dx); rel y = fmaf(c_i, dy, -(s_i * dx))
 *   O3  cos = fmaf(s_i, s_j, c_i * c_j); sin = fmaf(c_i, s_j, -(s_i * c_j)); length = 2 hx; width = 2 hy
 * Returns 0, or -1 on bad arguments. */
int orc_observe_vec(const orc_prim48 *prims, int P, int A, const float *speed, int K, int M, float radius,
                    int32_t *agent_idx, float *agent_feat, int32_t *road_idx, float *road_feat)
{
    if (!prims || !speed || A < 1 || P < A || K < 0 || M < 0) return -1;
    if ((K > 0 && (!agent_idx || !agent_feat)) || (M > 0 && (!road_idx || !road_feat))) return -1;
    const float r2 = radius * radius;
    for (int i = 0; i < A; ++i) {
        const orc_prim48 *e = &prims[i];
        /* ---- agents: K rounds of "smallest (d2, j) greater than the last one taken" */
        float last_d2 = -1.0f; int last_j = -1;
        for (int r = 0; r < K; ++r) {
            float best_d2 = 0.0f; int best_j = -1;
            for (int j = 0; j < A; ++j) {
                if (j == i) continue;
                float dx = prims[j].cx - e->cx, dy = prims[j].cy - e->cy;
                float d2 = fmaf(dy, dy, dx * dx);
                if (!(d2 <= r2)) continue;
                if (d2 < last_d2 || (d2 == last_d2 && j <= last_j)) continue;      /* already taken */
                if (best_j < 0 || d2 < best_d2) { best_d2 = d2; best_j = j; }       /* ascending j: first wins ties */
            }
            int32_t *oi = agent_idx + ((size_t)i * K + r);
            float *of = agent_feat + ((size_t)i * K + r) * 8;
            if (best_j < 0) {
                *oi = -1;
                for (int q = 0; q < 8; ++q) of[q] = 0.0f;
                last_d2 = INFINITY; last_j = A;                                     /* nothing further */
                continue;
            }
            const orc_prim48 *p = &prims[best_j];
            float dx = p->cx - e->cx, dy = p->cy - e->cy;
            *oi = best_j;
            of[0] = fmaf(e->sk, dy, e->ck * dx);
            of[1] = fmaf(e->ck, dy, -(e->sk * dx));
            of[2] = 2.0f * p->hx;
            of[3] = 2.0f * p->hy;
            of[4] = fmaf(e->sk, p->sk, e->ck * p->ck);
            of[5] = fmaf(e->ck, p->sk, -(e->sk * p->ck));
            of[6] = speed[best_j] - speed[i];
            of[7] = 1.0f;
            last_d2 = best_d2; last_j = best_j;
        }
        /* ---- road segments */
        last_d2 = -1.0f; last_j = -1;
        for (int r = 0; r < M; ++r) {
            float best_d2 = 0.0f; int best_j = -1;
            for (int k = A; k < P; ++k) {
                if (prims[k].shape != 0 || prims[k].hz != 0.0f) continue;           /* flat strips only */
                float dx = prims[k].cx - e->cx, dy = prims[k].cy - e->cy;
                float d2 = fmaf(dy, dy, dx * dx);
                if (!(d2 <= r2)) continue;
                if (d2 < last_d2 || (d2 == last_d2 && k <= last_j)) continue;
                if (best_j < 0 || d2 < best_d2) { best_d2 = d2; best_j = k; }
            }
            int32_t *oi = road_idx + ((size_t)i * M + r);
            float *of = road_feat + ((size_t)i * M + r) * 8;
            if (best_j < 0) {
                *oi = -1;
                for (int q = 0; q < 8; ++q) of[q] = 0.0f;
                last_d2 = INFINITY; last_j = P;
                continue;
            }
            const orc_prim48 *p = &prims[best_j];
            float dx = p->cx - e->cx, dy = p->cy - e->cy;
            *oi = best_j;
            of[0] = fmaf(e->sk, dy, e->ck * dx);
            of[1] = fmaf(e->ck, dy, -(e->sk * dx));
            of[2] = 2.0f * p->hx;
            of[3] = fmaf(e->sk, p->sk, e->ck * p->ck);
            of[4] = fmaf(e->ck, p->sk, -(e->sk * p->ck));
            of[5] = (float)p->cls;
            of[6] = 1.0f;
            of[7] = 0.0f;
            last_d2 = best_d2; last_j = best_j;
        }
    }
    return 0;
}
