// gp_kernel_sim.cuh — the step either side of the render: the jerk-actuated kinematic
// bicycle that advances the agents fused with the pose update a0, and the vectorised observation
// O_vec.  Contracts: DESIGN.md "Dynamics contract" D1-D6 (fp32 with libm atanf / tanf / sincosf:
// parity with the fp64 oracle by tolerance) and "Observation contract" O1-O3 (fp32 add / mul / fma only, explicit
// round-to-nearest intrinsics: bit-exact).
#pragma once
#include "gp_device.cuh"
#include "gp_kernels_basic.cuh"

namespace gp {

__device__ __forceinline__ float clipf(float x, float lo, float hi) { return fminf(fmaxf(x, lo), hi); }

// D1-D6 + a0.  One thread per agent: reads its action, kinematic state and pose, writes the new state and pose, the
// agent's primitive record (centre, heading) and its shading table, so the renderer can be called right after with
// no host transfer and no separate pose-update launch.
__global__ void k_dynamics_step(SceneConst sc, gp_dyn_params par, const int32_t *__restrict__ action,
                                float4 *__restrict__ state /* [n][2]: (v a_lon a_lat steer) (psi - - -) */,
                                float4 *__restrict__ pose, gp_prim *__restrict__ prims, PrimMeta *__restrict__ meta) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t n = (size_t)sc.Wn * sc.A;
    if (i >= n) return;
    const int a = __ldg(&action[i]);
    if (a < 0 || a >= 12) return;                                   // invalid action: the agent is left untouched
    const size_t w = i / sc.A, ag = i % sc.A;
    gp_prim *p = &prims[w * sc.P + ag];
    if (!(p->hx > 0.0f)) return;                                    // no length, no wheelbase (tan / L): left untouched too
    const float4 s0 = state[2 * i], s1 = state[2 * i + 1], ps = pose[i];
    const int il = a / 3, it = a - 3 * il;
    const float jlon = il == 0 ? -15.0f : il == 1 ? -4.0f : il == 2 ? 0.0f : 4.0f;
    const float jlat = it == 0 ? -4.0f : it == 1 ? 0.0f : 4.0f;
    const float dt = par.dt;
    float v = s0.x, a_lon = s0.y, a_lat = s0.z, steer = s0.w, psi = s1.x, x = ps.x, y = ps.y;
    a_lon = clipf(fmaf(jlon, dt, a_lon), -par.a_lon_max, par.a_lon_max);                 // D1
    a_lat = clipf(fmaf(jlat, dt, a_lat), -par.a_lat_max, par.a_lat_max);
    v = clipf(fmaf(a_lon, dt, v), 0.0f, par.v_max);                                      // D2
    const float L = 0.6f * (2.0f * p->hx);                                               // D3: wheelbase
    const float vv = fmaxf(v, par.v_eps);
    const float want = atanf(L * a_lat / (vv * vv));
    const float dmax = par.steer_rate_max * dt;
    steer = steer + clipf(want - steer, -dmax, dmax);
    steer = clipf(steer, -par.steer_max, par.steer_max);
    psi = fmaf(v * (tanf(steer) / L), dt, psi);                                          // D4
    const float PI = 3.14159265358979323846f;
    if (fabsf(psi) > 2.0f * PI) psi = remainderf(psi, 2.0f * PI);                        // more than a turn in one step (exact)
    if (psi >= PI) psi -= 2.0f * PI;
    if (psi < -PI) psi += 2.0f * PI;
    float sn, c;
    sincosf(psi, &sn, &c);
    x = fmaf(v * c, dt, x);                                                              // D5
    y = fmaf(v * sn, dt, y);
    if (par.extent > 0.0f) {                                                             // D6
        const float E = par.extent, h = 0.5f * E;
        if (x >= h) x -= E;
        if (x < -h) x += E;
        if (y >= h) y -= E;
        if (y < -h) y += E;
    }
    state[2 * i] = make_float4(v, a_lon, a_lat, steer);
    state[2 * i + 1] = make_float4(psi, s1.y, s1.z, s1.w);
    pose[i] = make_float4(x, y, c, sn);
    p->cx = x; p->cy = y; p->cos_yaw = c; p->sin_yaw = sn;                               // a0
    gp_prim q = *p;
    write_meta(q, &meta[w * sc.P + ag], sc);
}

// ---- O_vec -------------------------------------------------------------------------------------------------------
constexpr int kObsWarps = 8;                      // agents per CTA (one warp each), all of the same world
constexpr unsigned long long kObsNone = 0xFFFFFFFFFFFFFFFFull;

struct ObsArgs {
    int groups_per_world, K, M, nwarps;
    float r2;                                     // radius * radius (one fp32 product, formed on the host: O1)
    const float4 *state;                          // [Wn][A][2]; speed = .x of the first
    int32_t *agent_idx; float *agent_feat; int32_t *road_idx; float *road_feat;
};

// K (or M) rounds of "take the smallest remaining key": lanes scan the warp's key array in shared memory, a warp
// minimum picks the winner, its slot is struck out.  Keys are d2 bits << 32 | index (d2 >= 0: unsigned order = fp32
// order, ties by index: contract O1).  sel[r] = index taken in round r or -1.  General fallback (any n).
__device__ __forceinline__ void obs_select(unsigned long long *keys, int n, int rounds, int idx_base, int *sel, int lane) {
    for (int r = 0; r < rounds; ++r) {
        unsigned long long best = kObsNone;
        for (int q = lane; q < n; q += 32) best = min(best, keys[q]);
#pragma unroll
        for (int o = 16; o; o >>= 1) best = min(best, __shfl_xor_sync(0xffffffffu, best, o));
        const int idx = best == kObsNone ? -1 : (int)(uint32_t)best;
        if (lane == 0) {
            sel[r] = idx;
            if (idx >= 0) keys[idx - idx_base] = kObsNone;
        }
        __syncwarp();
    }
}

// The same selection for n <= 32 N candidates: every lane takes N keys (candidates lane, lane + 32, ...) into registers,
// sorts them once with a compile-time bitonic network and writes its sorted run back to its own slots of the warp's key
// array (which the host sizes to 32 (N + 1) slots: obs_key_slots).  The rounds are then a 32-way merge of the lanes' runs that
// keeps only each run's head in registers: warp minimum of the heads' d2 bits, then of the indices among the lanes that
// hold it (two REDUX; O1: lowest index first), and the one winning lane records its index and takes its next key from
// shared memory.  ~15 instructions per round, no branch; round 2 shifted the whole
// run down through 2 N registers per round instead (30 instructions; ncu: 65 % of the kernel's instructions).
template <int N>
__device__ __forceinline__ void obs_merge(unsigned long long *keys, int n, int rounds, int *sel, int lane) {
    unsigned long long k[N];
#pragma unroll
    for (int t = 0; t < N; ++t) { const int q = lane + 32 * t; k[t] = q < n ? keys[q] : kObsNone; }
#pragma unroll
    for (int size = 2; size <= N; size <<= 1)
#pragma unroll
        for (int stride = size >> 1; stride > 0; stride >>= 1)
#pragma unroll
            for (int i = 0; i < N; ++i) {
                const int j = i ^ stride;
                if (j > i) {
                    const bool up = (i & size) == 0;
                    const unsigned long long x = k[i], y = k[j];
                    const bool sw = up ? x > y : x < y;
                    k[i] = sw ? y : x; k[j] = sw ? x : y;
                }
            }
    // rounds beyond the number of candidates within the radius are padding: count them once instead of testing every round
    int valid = 0;
#pragma unroll
    for (int t = 0; t < N; ++t) valid += (uint32_t)(k[t] >> 32) != 0xffffffffu;      // d2 bits < 0x7f800000: all ones = "none"
    const int live = min(rounds, (int)__reduce_add_sync(0xffffffffu, (unsigned)valid));
#pragma unroll
    for (int t = 1; t < N; ++t) keys[lane + 32 * t] = k[t];                  // the run behind the head, in the lane's own slots
    keys[lane + 32 * N] = kObsNone;                                          // ... closed by a sentinel (no bound test per round)
    uint32_t hi = (uint32_t)(k[0] >> 32), lo = (uint32_t)k[0];
    const unsigned long long *next = keys + lane + 32;                       // the key behind the head
    uint32_t sel_addr = (uint32_t)__cvta_generic_to_shared(sel);
    for (int r = 0; r < live; ++r, sel_addr += 4) {
        // two dependent warp minima, no branch: the smallest d2 among the heads, then the lowest index among the lanes that
        // hold it (O1; exactly one lane wins).  A ballot + "more than one bit?" test would save the second REDUX in the
        // common case, but costs a branch and a convergence barrier per round (measured: 24 instructions per round against 15)
        const uint32_t mh = __reduce_min_sync(0xffffffffu, hi);
        const uint32_t ml = __reduce_min_sync(0xffffffffu, hi == mh ? lo : 0xffffffffu);
        const bool win = hi == mh && lo == ml;
        const unsigned long long nx = *next;                                 // every lane reads; only the winner takes it
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %0, 0;\n\t@p st.shared.u32 [%1], %2;\n\t}"
                     :: "r"((unsigned)win), "r"(sel_addr), "r"(lo) : "memory");
        hi = win ? (uint32_t)(nx >> 32) : hi;
        lo = win ? (uint32_t)nx : lo;
        next += win ? 32 : 0;
    }
    for (int q = live + lane; q < rounds; q += 32) sel[q] = -1;
    __syncwarp();
}

// Slots of the per-warp key array for n candidates (host and device agree): 32 (N + 1) for the register-sorted merge.
__host__ __device__ inline int obs_key_slots(int n) {
    return n <= 64 ? 96 : n <= 128 ? 160 : n <= 256 ? 288 : n <= 512 ? 544 : n;      // 32 N run slots + 32 sentinels
}

__device__ __forceinline__ void obs_pick(unsigned long long *keys, int n, int rounds, int idx_base, int *sel, int lane) {
    if (n <= 64) obs_merge<2>(keys, n, rounds, sel, lane);
    else if (n <= 128) obs_merge<4>(keys, n, rounds, sel, lane);
    else if (n <= 256) obs_merge<8>(keys, n, rounds, sel, lane);
    else if (n <= 512) obs_merge<16>(keys, n, rounds, sel, lane);
    else obs_select(keys, n, rounds, idx_base, sel, lane);
}

// Grid: one CTA per (world, group of nwarps agents).  Dynamic shared memory: float4 s_a[P] (x, y, cos, sin),
// float4 s_b[P] (2 hx, 2 hy, speed | cls, road flag), unsigned long long s_keys[nwarps][obs_key_slots(max(A, Q))],
// int s_sel[nwarps][max(K, M)].
__global__ void __launch_bounds__(kObsWarps * 32)
k_observe_vec(SceneConst sc, ObsArgs oa, const gp_prim *__restrict__ prims) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int P = sc.P, A = sc.A, Q = sc.Q;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nmax = obs_key_slots(max(A, Q)), rmax = max(oa.K, oa.M);
    float4 *s_a = reinterpret_cast<float4 *>(smem);
    float4 *s_b = s_a + P;
    unsigned long long *s_keys = reinterpret_cast<unsigned long long *>(s_b + P) + (size_t)warp * nmax;
    int *s_sel = reinterpret_cast<int *>(reinterpret_cast<unsigned long long *>(s_b + P) + (size_t)oa.nwarps * nmax) + warp * rmax;
    const int w = blockIdx.x / oa.groups_per_world;
    const int i = (blockIdx.x - w * oa.groups_per_world) * oa.nwarps + warp;       // agent
    const gp_prim *wp = prims + (size_t)w * P;
    for (int k = threadIdx.x; k < P; k += blockDim.x) {
        const float4 *rec = reinterpret_cast<const float4 *>(&wp[k]);
        const float4 p0 = __ldg(rec), p1 = __ldg(rec + 1), p2 = __ldg(rec + 2);    // cx cy cz hx | hy hz ck sk | cls inst shape pad
        s_a[k] = make_float4(p0.x, p0.y, p1.z, p1.w);
        const bool road = k >= A && __float_as_int(p2.z) == GP_SHAPE_BOX && p1.y == 0.0f;     // flat strips only
        const float third = k < A ? __ldg(&oa.state[2 * ((size_t)w * A + k)]).x : (float)__float_as_int(p2.x);
        s_b[k] = make_float4(c_mul(2.0f, p0.w), c_mul(2.0f, p1.x), third, road ? 1.0f : 0.0f);
    }
    __syncthreads();
    if (i >= A) return;
    const float4 e = s_a[i];
    const float ev = s_b[i].z;
    const size_t ai = (size_t)w * A + i;
    // ---- surrounding agents -----------------------------------------------------------------------
    if (oa.K > 0) {
        for (int j = lane; j < A; j += 32) {
            const float4 q = s_a[j];
            const float dx = c_sub(q.x, e.x), dy = c_sub(q.y, e.y);
            const float d2 = c_fma(dy, dy, c_mul(dx, dx));                                      // O1
            s_keys[j] = (j != i && d2 <= oa.r2) ? ((unsigned long long)__float_as_uint(d2) << 32) | (uint32_t)j : kObsNone;
        }
        __syncwarp();
        obs_pick(s_keys, A, oa.K, 0, s_sel, lane);
        for (int r = lane; r < oa.K; r += 32) {
            const int j = s_sel[r];
            float4 f0 = make_float4(0.f, 0.f, 0.f, 0.f), f1 = f0;
            if (j >= 0) {
                const float4 q = s_a[j], b = s_b[j];
                const float dx = c_sub(q.x, e.x), dy = c_sub(q.y, e.y);
                f0 = make_float4(c_fma(e.w, dy, c_mul(e.z, dx)), c_fma(e.z, dy, -c_mul(e.w, dx)), b.x, b.y);        // O2
                f1 = make_float4(c_fma(e.w, q.w, c_mul(e.z, q.z)), c_fma(e.z, q.w, -c_mul(e.w, q.z)), c_sub(b.z, ev), 1.0f);   // O3
            }
            oa.agent_idx[ai * oa.K + r] = j;
            float4 *o = reinterpret_cast<float4 *>(oa.agent_feat + (ai * oa.K + r) * 8);
            o[0] = f0; o[1] = f1;
        }
        __syncwarp();
    }
    // ---- road segments ----------------------------------------------------------------------------
    if (oa.M > 0) {
        for (int k = lane; k < Q; k += 32) {
            const float4 q = s_a[A + k];
            const float dx = c_sub(q.x, e.x), dy = c_sub(q.y, e.y);
            const float d2 = c_fma(dy, dy, c_mul(dx, dx));
            s_keys[k] = (s_b[A + k].w != 0.0f && d2 <= oa.r2) ? ((unsigned long long)__float_as_uint(d2) << 32) | (uint32_t)(A + k) : kObsNone;
        }
        __syncwarp();
        obs_pick(s_keys, Q, oa.M, A, s_sel, lane);
        for (int r = lane; r < oa.M; r += 32) {
            const int k = s_sel[r];
            float4 f0 = make_float4(0.f, 0.f, 0.f, 0.f), f1 = f0;
            if (k >= 0) {
                const float4 q = s_a[k], b = s_b[k];
                const float dx = c_sub(q.x, e.x), dy = c_sub(q.y, e.y);
                f0 = make_float4(c_fma(e.w, dy, c_mul(e.z, dx)), c_fma(e.z, dy, -c_mul(e.w, dx)), b.x,
                                 c_fma(e.w, q.w, c_mul(e.z, q.z)));
                f1 = make_float4(c_fma(e.z, q.w, -c_mul(e.w, q.z)), b.z, 1.0f, 0.0f);
            }
            oa.road_idx[ai * oa.M + r] = k;
            float4 *o = reinterpret_cast<float4 *>(oa.road_feat + (ai * oa.M + r) * 8);
            o[0] = f0; o[1] = f1;
        }
    }
}

}  // namespace gp
