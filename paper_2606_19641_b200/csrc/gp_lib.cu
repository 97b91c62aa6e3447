// gp_lib.cu — the C ABI of include/gp.h on top of the sm_100a kernels.  Host logic only: argument
// validation, device residency of the scene, scratch sizing, launches.  No CPU rendering path exists.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "gp_device.cuh"
#include "gp_kernels_basic.cuh"
#include "gp_kernel_cull.cuh"
#include "gp_kernel_render.cuh"
#include "gp_kernel_raster.cuh"
#include "gp_kernel_sim.cuh"
#include "gp_kernel_probe.cuh"

using namespace gp;

#ifndef GP_TINY_PX
#define GP_TINY_PX 1024            // images of up to this many pixels are rendered by one-warp CTAs (plan_render)
#endif
#ifndef GP_STAGE_CAP
#define GP_STAGE_CAP 128
#endif

struct gp_ctx {
    int device = -1;
    bool have_scene = false, has_spheres = false;     // has_spheres: the uploaded records held a sphere
    bool statics_touched = false;                     // gp_statics_update ran since the upload (may have added spheres)
    SceneConst sc{};
    gp_prim *d_prims = nullptr;
    PrimMeta *d_meta = nullptr;
    float2 *d_pitch = nullptr;
    gp_prim *h_stage = nullptr; size_t h_stage_bytes = 0;        // pinned upload staging
    // per-view scratch of the fast path
    ViewHdr *d_hdr = nullptr; EntryGeo *d_geo = nullptr; EntryAux *d_aux = nullptr;
    uint8_t *d_ovf = nullptr;                                    // per view: its list did not fit GP_OPT_LIST_CAP
    size_t scratch_views = 0; int scratch_cap = 0;
    unsigned long long *d_stats = nullptr;                      // [0..1] GP_OPT_STATS counters, [2..3] scratch of gp_probe
    int n_sms = 148;
    int opt_path = GP_PATH_FAST, opt_stats = 0, opt_timing = 0, opt_stage_cap = 0, opt_strip_px = 0, opt_gather = -1, opt_spheres = -1;
    int opt_variant = -1, opt_tile_px = 0, opt_pipeline = 1, opt_list_cap = 0;
    cudaStream_t aux_stream = nullptr;                           // culls of later chunks run here (render_device)
    std::vector<cudaEvent_t> pipe_ev;
    struct Timed { int kernel; cudaEvent_t a, b; };
    std::vector<Timed> timed;                                    // GP_OPT_TIMING records
    std::vector<cudaEvent_t> ev_pool;
    uint64_t launches = 0;
    unsigned timing_seq[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    size_t obs_smem_set = 0;
    int last_H = 0, last_W = 0;                                  // image size of the last gp_render_batch (GP_PROBE_STORE_VIEW)
    size_t render_smem_set = 0, raster_smem_set = 0;
    // gp_render_batch_host staging
    float *d_pose = nullptr;
    unsigned char *d_out[2] = {nullptr, nullptr}; size_t d_out_bytes = 0;
    cudaStream_t copy_stream = nullptr; cudaEvent_t ev_render[2] = {nullptr, nullptr}, ev_copy[2] = {nullptr, nullptr};
};

static thread_local char g_cuda_msg[256] = "CUDA error";

static int cuda_fail(cudaError_t e, const char *where) {
    snprintf(g_cuda_msg, sizeof g_cuda_msg, "CUDA error at %s: %s", where, cudaGetErrorString(e));
    return GP_ERR_CUDA;
}
#define CK(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, #call); } while (0)

// Brackets one kernel launch with events when GP_OPT_TIMING is on.  At most kMaxTimed records are kept.
constexpr size_t kMaxTimed = 4096;
struct LaunchTimer {
    gp_ctx *c; cudaStream_t s; bool on; gp_ctx::Timed t{};
    LaunchTimer(gp_ctx *c_, int kernel, cudaStream_t s_) : c(c_), s(s_), on(false) {
        if (c->opt_timing <= 0) return;
        cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;              // no event records inside a graph capture
        if (cudaStreamIsCapturing(s, &cap) != cudaSuccess) { cudaGetLastError(); return; }
        if (cap != cudaStreamCaptureStatusNone) return;
        on = (c->timing_seq[kernel & 7]++ % (unsigned)c->opt_timing) == 0;     // every opt_timing-th launch of this kernel
        if (!on) return;
        if (c->timed.size() >= kMaxTimed) {                                     // never polled: recycle the oldest record
            c->ev_pool.push_back(c->timed.front().a); c->ev_pool.push_back(c->timed.front().b);
            c->timed.erase(c->timed.begin());
        }
        t.kernel = kernel;
        cudaEvent_t *e[2] = {&t.a, &t.b};
        for (auto p : e) {
            if (!c->ev_pool.empty()) { *p = c->ev_pool.back(); c->ev_pool.pop_back(); }
            else if (cudaEventCreate(p) != cudaSuccess) { on = false; return; }
        }
        cudaEventRecord(t.a, s);
    }
    ~LaunchTimer() { if (on) { cudaEventRecord(t.b, s); c->timed.push_back(t); } }
};

static bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// Every ABI entry runs on the context's device, whatever device the calling thread had current, and leaves the
// caller's current device as it found it.
struct DeviceGuard {
    int prev = -1; bool ok = true;
    explicit DeviceGuard(const gp_ctx *c) {
        if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; cudaGetLastError(); }
        if (prev != c->device) ok = cudaSetDevice(c->device) == cudaSuccess; else prev = -1;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define GP_ON_DEVICE(c) DeviceGuard guard_(c); if (!guard_.ok) return cuda_fail(cudaGetLastError(), "cudaSetDevice")

extern "C" const char *gp_error_string(int code) {
    switch (code) {
        case GP_OK: return "ok";
        case GP_ERR_ARG: return "invalid argument";
        case GP_ERR_ALIGN: return "pointer not 16-byte aligned";
        case GP_ERR_STATE: return "no scene uploaded";
        case GP_ERR_RANGE: return "world range or agent count outside the scene";
        case GP_ERR_CUDA: return g_cuda_msg;
        case GP_ERR_ARCH: return "device is not sm_100 (B200); no fallback path exists";
        case GP_ERR_NOMEM: return "out of memory";
        case GP_ERR_LIMIT: return "gp_render_static: the scene exceeds GP_STATIC_MAX_VIEWS / _PRIMS / _ENTRIES (its scratch "
                                  "is a fixed array; render fewer worlds per call or use a gp_ctx)";
        default: return "unknown error code";
    }
}

extern "C" int gp_create(gp_ctx **out, int cuda_device) {
    if (!out) return GP_ERR_ARG;
    *out = nullptr;
    int count = 0;
    CK(cudaGetDeviceCount(&count));
    if (cuda_device < 0 || cuda_device >= count) return GP_ERR_ARG;
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, cuda_device));
    if (prop.major != 10) return GP_ERR_ARCH;
    CK(cudaSetDevice(cuda_device));
    gp_ctx *c = new (std::nothrow) gp_ctx();
    if (!c) return GP_ERR_NOMEM;
    c->device = cuda_device;
    c->sc.C = 1;                                                   // default rig: one front camera
    c->sc.rig[0] = make_float4(1.0f, 0.0f, 1.0f, 0.0f);
    c->n_sms = prop.multiProcessorCount;
    cudaError_t e = cudaMalloc(&c->d_stats, 4 * sizeof(unsigned long long));
    if (e != cudaSuccess) { delete c; return cuda_fail(e, "cudaMalloc(stats)"); }
    cudaMemset(c->d_stats, 0, 4 * sizeof(unsigned long long));
    *out = c;
    return GP_OK;
}

static void free_scene(gp_ctx *c) {
    cudaFree(c->d_prims); cudaFree(c->d_meta); cudaFree(c->d_pitch);
    c->d_prims = nullptr; c->d_meta = nullptr; c->d_pitch = nullptr;
    cudaFree(c->d_hdr); cudaFree(c->d_geo); cudaFree(c->d_aux); cudaFree(c->d_ovf);
    c->d_hdr = nullptr; c->d_geo = nullptr; c->d_aux = nullptr; c->d_ovf = nullptr; c->scratch_views = 0; c->scratch_cap = 0;
    cudaFree(c->d_pose); c->d_pose = nullptr;
    c->have_scene = false;
}

extern "C" int gp_destroy(gp_ctx *c) {
    if (!c) return GP_ERR_ARG;
    {
    GP_ON_DEVICE(c);
    cudaDeviceSynchronize();
    free_scene(c);
    for (int i = 0; i < 2; ++i) {
        cudaFree(c->d_out[i]);
        if (c->ev_render[i]) cudaEventDestroy(c->ev_render[i]);
        if (c->ev_copy[i]) cudaEventDestroy(c->ev_copy[i]);
    }
    for (auto &t : c->timed) { cudaEventDestroy(t.a); cudaEventDestroy(t.b); }
    for (auto e : c->ev_pool) cudaEventDestroy(e);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->aux_stream) cudaStreamDestroy(c->aux_stream);
    for (auto e : c->pipe_ev) cudaEventDestroy(e);
    if (c->h_stage) cudaFreeHost(c->h_stage);
    cudaFree(c->d_stats);
    }
    delete c;
    return GP_OK;
}

extern "C" int gp_set_option(gp_ctx *c, int key, int value) {
    if (!c) return GP_ERR_ARG;
    switch (key) {
        case GP_OPT_PATH:
            if (value != GP_PATH_FAST && value != GP_PATH_BRUTE) return GP_ERR_ARG;
            c->opt_path = value; return GP_OK;
        case GP_OPT_STATS:
            c->opt_stats = value ? 1 : 0; return GP_OK;
        case GP_OPT_TIMING:
            if (value < 0) return GP_ERR_ARG;
            c->opt_timing = value;
            for (unsigned &q : c->timing_seq) q = 0;
            return GP_OK;
        case GP_OPT_STAGE_CAP:
            if (value < 0) return GP_ERR_ARG;
            c->opt_stage_cap = value; return GP_OK;
        case GP_OPT_GATHER:
            if (value < -1 || value > 1) return GP_ERR_ARG;
            c->opt_gather = value; return GP_OK;
        case GP_OPT_VARIANT:
            if (value < -1 || value > GP_VARIANT_RASTER) return GP_ERR_ARG;
            c->opt_variant = value; return GP_OK;
        case GP_OPT_PIPELINE:
            if (value < 1 || value > 64) return GP_ERR_ARG;
            c->opt_pipeline = value; return GP_OK;
        case GP_OPT_TILE_PX:
            if (value < 0 || value > 16384) return GP_ERR_ARG;
            c->opt_tile_px = value; return GP_OK;
        case GP_OPT_SPHERES:
            if (value < -1 || value > 1) return GP_ERR_ARG;
            c->opt_spheres = value; return GP_OK;
        case GP_OPT_LIST_CAP:
            if (value < 0) return GP_ERR_ARG;
            c->opt_list_cap = value; return GP_OK;
        case GP_OPT_STRIP_PX:
            if (value < 0 || value > 4096) return GP_ERR_ARG;
            c->opt_strip_px = value; return GP_OK;
        default: return GP_ERR_ARG;
    }
}

extern "C" int gp_scene_upload(gp_ctx *c, const gp_scene_desc *d, const gp_prim *h_agents,
                               const gp_prim *h_quads, void *stream_) {
    if (!c || !d || !h_agents) return GP_ERR_ARG;
    if (d->n_worlds < 1 || d->agents_per_world < 1 || d->quads_per_world < 0) return GP_ERR_ARG;
    if (d->quads_per_world > 0 && !h_quads) return GP_ERR_ARG;
    if (!(d->cam_height > 0.0f) || !(d->t_max > 0.0f) || !(d->ambient >= 0.0f && d->ambient <= 1.0f)) return GP_ERR_ARG;
    const long long P = (long long)d->agents_per_world + d->quads_per_world;
    if (P >= (1 << 19) || (long long)d->n_worlds * P > (1ll << 31)) return GP_ERR_ARG;
    const size_t Wn = d->n_worlds, A = d->agents_per_world, Q = d->quads_per_world, n = Wn * (size_t)P;
    for (size_t i = 0; i < Wn * A; ++i) {
        const gp_prim &p = h_agents[i];
        if (p.cls < 0 || p.cls > 7 || (p.shape != GP_SHAPE_BOX && p.shape != GP_SHAPE_SPHERE) ||
            !(p.hx >= 0.0f && p.hy >= 0.0f && p.hz >= 0.0f)) return GP_ERR_ARG;
    }
    for (size_t i = 0; i < Wn * Q; ++i) {
        const gp_prim &p = h_quads[i];
        if (p.cls < 0 || p.cls > 7 || (p.shape != GP_SHAPE_BOX && p.shape != GP_SHAPE_SPHERE) ||
            !(p.hx >= 0.0f && p.hy >= 0.0f && p.hz >= 0.0f)) return GP_ERR_ARG;
    }
    bool spheres = false;
    for (size_t i = 0; i < Wn * A; ++i) spheres |= h_agents[i].shape == GP_SHAPE_SPHERE;
    for (size_t i = 0; i < Wn * Q; ++i) spheres |= h_quads[i].shape == GP_SHAPE_SPHERE;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    GP_ON_DEVICE(c);
    CK(cudaDeviceSynchronize());            // earlier work may still read the old scene
    free_scene(c);
    if (c->h_stage_bytes < n * sizeof(gp_prim)) {
        if (c->h_stage) cudaFreeHost(c->h_stage);
        c->h_stage = nullptr; c->h_stage_bytes = 0;
        if (cudaMallocHost(&c->h_stage, n * sizeof(gp_prim)) != cudaSuccess) { cudaGetLastError(); return GP_ERR_NOMEM; }
        c->h_stage_bytes = n * sizeof(gp_prim);
    }
    for (size_t w = 0; w < Wn; ++w) {       // interleave into one table [Wn][A+Q]
        memcpy(c->h_stage + w * P, h_agents + w * A, A * sizeof(gp_prim));
        if (Q) memcpy(c->h_stage + w * P + A, h_quads + w * Q, Q * sizeof(gp_prim));
    }
    if (cudaMalloc(&c->d_prims, n * sizeof(gp_prim)) != cudaSuccess ||
        cudaMalloc(&c->d_meta, n * sizeof(PrimMeta)) != cudaSuccess ||
        cudaMalloc(&c->d_pitch, Wn * A * sizeof(float2)) != cudaSuccess ||
        cudaMalloc(&c->d_pose, Wn * A * 4 * sizeof(float)) != cudaSuccess) {
        cudaGetLastError(); free_scene(c); return GP_ERR_NOMEM;
    }
    SceneConst &sc = c->sc;
    sc.Wn = (int)Wn; sc.A = (int)A; sc.Q = (int)Q; sc.P = (int)P;
    sc.cam_h = d->cam_height; sc.t_max = d->t_max;
    sc.Lx = d->light[0]; sc.Ly = d->light[1]; sc.Lz = d->light[2]; sc.ambient = d->ambient;
    for (int k = 0; k < 8; ++k)
        sc.pal[k] = (uint32_t)d->palette[k][0] | ((uint32_t)d->palette[k][1] << 8) | ((uint32_t)d->palette[k][2] << 16);
    CK(cudaMemcpyAsync(c->d_prims, c->h_stage, n * sizeof(gp_prim), cudaMemcpyHostToDevice, stream));
    k_prim_meta<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(sc, c->d_prims, c->d_meta);
    k_fill_pitch<<<(unsigned)((Wn * A + 255) / 256), 256, 0, stream>>>(c->d_pitch, Wn * A);
    c->launches += 2;
    CK(cudaGetLastError());
    c->have_scene = true;
    c->has_spheres = spheres;
    c->statics_touched = false;
    return GP_OK;
}

extern "C" int gp_agents_update(gp_ctx *c, const float *d_pose, void *stream_) {
    if (!c || !d_pose) return GP_ERR_ARG;
    if (!c->have_scene) return GP_ERR_STATE;
    if (!aligned16(d_pose)) return GP_ERR_ALIGN;
    GP_ON_DEVICE(c);
    const size_t n = (size_t)c->sc.Wn * c->sc.A;
    {
        LaunchTimer lt(c, GP_KERNEL_UPDATE, static_cast<cudaStream_t>(stream_));
        k_agents_update<<<(unsigned)((n + 255) / 256), 256, 0, static_cast<cudaStream_t>(stream_)>>>(
            c->sc, reinterpret_cast<const float4 *>(d_pose), c->d_prims, c->d_meta);
    }
    c->launches += 1;
    CK(cudaGetLastError());
    return GP_OK;
}

extern "C" int gp_dynamics_step(gp_ctx *c, const gp_dyn_params *par, const int32_t *d_action, float *d_state,
                                float *d_pose, void *stream_) {
    if (!c || !par || !d_action || !d_state || !d_pose) return GP_ERR_ARG;
    if (!c->have_scene) return GP_ERR_STATE;
    if (!(par->dt > 0.0f) || !(par->a_lon_max >= 0.0f) || !(par->a_lat_max >= 0.0f) || !(par->v_max >= 0.0f) ||
        !(par->steer_max >= 0.0f) || !(par->steer_rate_max >= 0.0f) || !(par->v_eps > 0.0f) || !(par->extent >= 0.0f))
        return GP_ERR_ARG;
    if (!(par->steer_max < 1.5707f)) return GP_ERR_ARG;             // tan(steer) must stay finite
    if (!aligned16(d_state) || !aligned16(d_pose)) return GP_ERR_ALIGN;
    GP_ON_DEVICE(c);
    const size_t n = (size_t)c->sc.Wn * c->sc.A;
    {
        LaunchTimer lt(c, GP_KERNEL_DYNAMICS, static_cast<cudaStream_t>(stream_));
        k_dynamics_step<<<(unsigned)((n + 127) / 128), 128, 0, static_cast<cudaStream_t>(stream_)>>>(
            c->sc, *par, d_action, reinterpret_cast<float4 *>(d_state), reinterpret_cast<float4 *>(d_pose), c->d_prims, c->d_meta);
    }
    c->launches += 1;
    CK(cudaGetLastError());
    return GP_OK;
}

extern "C" int gp_observe_vec(gp_ctx *c, const float *d_state, int K, int M, float radius, int32_t *d_agent_idx,
                              float *d_agent_feat, int32_t *d_road_idx, float *d_road_feat, void *stream_) {
    if (!c || !d_state || K < 0 || M < 0 || K > 1024 || M > 1024 || (K == 0 && M == 0) || !(radius >= 0.0f)) return GP_ERR_ARG;
    if ((K > 0 && (!d_agent_idx || !d_agent_feat)) || (M > 0 && (!d_road_idx || !d_road_feat))) return GP_ERR_ARG;
    if (!c->have_scene) return GP_ERR_STATE;
    if (!aligned16(d_state) || !aligned16(d_agent_feat) || !aligned16(d_road_feat)) return GP_ERR_ALIGN;
    GP_ON_DEVICE(c);
    const SceneConst &sc = c->sc;
    ObsArgs oa;
    oa.K = K; oa.M = M; oa.r2 = radius * radius;
    oa.state = reinterpret_cast<const float4 *>(d_state);
    oa.agent_idx = d_agent_idx; oa.agent_feat = d_agent_feat; oa.road_idx = d_road_idx; oa.road_feat = d_road_feat;
    // agents per CTA: as many warps (<= kObsWarps) as leave the world's records + per-warp key arrays within shared memory
    const size_t nmax = (size_t)obs_key_slots(std::max(sc.A, sc.Q)), rmax = (size_t)std::max(K, M);
    int nw = std::min(kObsWarps, sc.A);
    size_t smem = 0;
    for (;; --nw) {
        smem = (size_t)sc.P * 32 + (size_t)nw * nmax * 8 + (size_t)nw * rmax * 4;
        if (smem <= 200 * 1024 || nw == 1) break;
    }
    if (smem > 200 * 1024) return GP_ERR_ARG;
    oa.nwarps = nw; oa.groups_per_world = (sc.A + nw - 1) / nw;
    if (smem > c->obs_smem_set) {
        CK(cudaFuncSetAttribute(k_observe_vec, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        c->obs_smem_set = smem;
    }
    {
        LaunchTimer lt(c, GP_KERNEL_OBSERVE, static_cast<cudaStream_t>(stream_));
        k_observe_vec<<<(unsigned)((size_t)sc.Wn * oa.groups_per_world), nw * 32, smem, static_cast<cudaStream_t>(stream_)>>>(sc, oa, c->d_prims);
    }
    c->launches += 1;
    CK(cudaGetLastError());
    return GP_OK;
}

extern "C" int gp_statics_update(gp_ctx *c, const gp_prim *d_prims, int n, int q_begin, void *stream_) {
    if (!c || !d_prims || n < 1) return GP_ERR_ARG;
    if (!c->have_scene) return GP_ERR_STATE;
    if (!aligned16(d_prims)) return GP_ERR_ALIGN;
    if (q_begin < 0 || (long long)q_begin + n > c->sc.Q) return GP_ERR_RANGE;
    GP_ON_DEVICE(c);
    c->statics_touched = true;      // the records are device memory the host never sees: they may hold spheres
    const size_t total = (size_t)c->sc.Wn * n;
    k_statics_update<<<(unsigned)((total + 255) / 256), 256, 0, static_cast<cudaStream_t>(stream_)>>>(
        c->sc, d_prims, n, q_begin, c->d_prims, c->d_meta);
    c->launches += 1;
    CK(cudaGetLastError());
    return GP_OK;
}

extern "C" int gp_statics_from_polylines(gp_ctx *c, const float *d_points, int n_lines, int pts_per_line,
                                         float half_width, float z, int cls, int q_begin, void *stream_) {
    if (!c || !d_points) return GP_ERR_ARG;
    if (!c->have_scene) return GP_ERR_STATE;
    if (n_lines < 1 || pts_per_line < 2 || cls < 0 || cls > 7 || !(half_width >= 0.0f)) return GP_ERR_ARG;
    if (reinterpret_cast<uintptr_t>(d_points) & 7u) return GP_ERR_ALIGN;
    const long long per_world = (long long)n_lines * (pts_per_line - 1);
    if (q_begin < 0 || q_begin + per_world > c->sc.Q) return GP_ERR_RANGE;
    GP_ON_DEVICE(c);
    const size_t n = (size_t)c->sc.Wn * (size_t)per_world;
    k_polyline_quads<<<(unsigned)((n + 255) / 256), 256, 0, static_cast<cudaStream_t>(stream_)>>>(
        c->sc, reinterpret_cast<const float2 *>(d_points), n_lines, pts_per_line, half_width, z, cls, q_begin,
        c->d_prims, c->d_meta);
    c->launches += 1;
    CK(cudaGetLastError());
    return GP_OK;
}

extern "C" int gp_cameras_set(gp_ctx *c, const float *d_pitch_cs, void *stream_) {
    if (!c) return GP_ERR_ARG;
    if (!c->have_scene) return GP_ERR_STATE;
    GP_ON_DEVICE(c);
    const size_t n = (size_t)c->sc.Wn * c->sc.A;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    if (d_pitch_cs) {
        CK(cudaMemcpyAsync(c->d_pitch, d_pitch_cs, n * sizeof(float2), cudaMemcpyDeviceToDevice, stream));
    } else {
        k_fill_pitch<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(c->d_pitch, n);
        c->launches += 1;
        CK(cudaGetLastError());
    }
    return GP_OK;
}

extern "C" int gp_camera_rig_set(gp_ctx *c, int n_cams, const gp_camera *h_rig) {
    if (!c || !h_rig || n_cams < 1 || n_cams > GP_MAX_CAMS) return GP_ERR_ARG;
    for (int i = 0; i < n_cams; ++i) {
        const gp_camera &q = h_rig[i];
        if (!(fabsf(q.cos_yaw_off) <= 1.0f && fabsf(q.sin_yaw_off) <= 1.0f && fabsf(q.mount) <= 16.0f)) return GP_ERR_ARG;
    }
    c->sc.C = n_cams;
    for (int i = 0; i < n_cams; ++i)
        c->sc.rig[i] = make_float4(h_rig[i].cos_yaw_off, h_rig[i].sin_yaw_off, h_rig[i].mount, 0.0f);
    return GP_OK;
}

// Per-view scratch of the fast path: header + list of up to `cap` entries per view, cap = P (every primitive of the world could be
// listed) unless GP_OPT_LIST_CAP sets a smaller one; then a view whose list does not fit is flagged in d_ovf and rendered by
// the brute-force kernel after the render pass (render_device), so the result stays the all-primitive definition.
static int list_cap(const gp_ctx *c) {
    return c->opt_list_cap > 0 ? std::min(c->sc.P, c->opt_list_cap) : c->sc.P;
}
static int ensure_scratch(gp_ctx *c, size_t views) {
    const int cap = list_cap(c);
    if (c->scratch_views >= views && c->scratch_cap == cap) return GP_OK;
    CK(cudaDeviceSynchronize());
    cudaFree(c->d_hdr); cudaFree(c->d_geo); cudaFree(c->d_aux); cudaFree(c->d_ovf);
    c->d_hdr = nullptr; c->d_geo = nullptr; c->d_aux = nullptr; c->d_ovf = nullptr; c->scratch_views = 0;
    if (cudaMalloc(&c->d_hdr, views * sizeof(ViewHdr)) != cudaSuccess ||
        cudaMalloc(&c->d_geo, views * cap * sizeof(EntryGeo)) != cudaSuccess ||
        cudaMalloc(&c->d_aux, views * cap * sizeof(EntryAux)) != cudaSuccess ||
        cudaMalloc(&c->d_ovf, views) != cudaSuccess) {
        cudaGetLastError();
        cudaFree(c->d_hdr); cudaFree(c->d_geo); cudaFree(c->d_aux); cudaFree(c->d_ovf);
        c->d_hdr = nullptr; c->d_geo = nullptr; c->d_aux = nullptr; c->d_ovf = nullptr;
        return GP_ERR_NOMEM;
    }
    c->scratch_views = views; c->scratch_cap = cap;
    return GP_OK;
}

static int check_render_args(gp_ctx *c, int world_begin, int n_worlds, int agents, int H, int W, float fov) {
    if (!c) return GP_ERR_ARG;
    if (!c->have_scene) return GP_ERR_STATE;
    if (H < 1 || W < 1 || H > 4096 || W > 4096 || n_worlds < 1 || world_begin < 0) return GP_ERR_ARG;
    if (!(fov > 0.0f && fov < 3.1415f)) return GP_ERR_ARG;
    if (agents != c->sc.A || (long long)world_begin + n_worlds > c->sc.Wn) return GP_ERR_RANGE;
    return GP_OK;
}

// Launch shape of the render pass for an H x W image (host logic; all thresholds measured on B200).
struct RenderPlan { int SR, log2LC, log2W, ng, ngr, nwarps, gather, scap; uint32_t magicW; size_t smem; };
static bool plan_render(const gp_ctx *c, const SceneConst &sc, int H, int W, RenderPlan &pl) {
    // List entries staged in shared memory (longer lists read their tail from global memory): 128; 64 for images of up to
    // 64 x 64 pixels, whose CTAs are small enough for the list buffer to decide how many fit an SM (measured: small 0.1072 ->
    // 0.1026 ms, sweep 64 x 64 0.381 -> 0.348 ms; 210 x 126 and larger lose with 64)
    // (48 for images of up to 32 x 32, rendered by one-warp CTAs of which 32 then fit an SM)
    const bool tiny = (long long)H * W <= GP_TINY_PX;
    pl.scap = std::min(sc.P, c->opt_stage_cap > 0 ? c->opt_stage_cap : tiny ? 48 : (long long)H * W <= 64 * 64 ? 64 : GP_STAGE_CAP);
    // rows per strip (power of two): ~512 pixels, fewer for small images so that a view still has
    // >= 8 strips to spread over its warps (a strip's entries are processed serially by one warp; measured: 64 x 64 with
    // 8 strips of 512 pixels 0.1072 ms against 0.1135 with 16 of 256 on the small configuration, equal on the sweep's)
    int strip_px = c->opt_strip_px;
    if (strip_px <= 0) { strip_px = 512; while (strip_px > 128 && H * W / strip_px < 8) strip_px /= 2; }
    // Images of up to 32 x 32: ONE warp per view and strips of 256 pixels (measured on the sweep's 32 x 32: 0.148 ms against
    // 0.166 with 2 warps and 128-pixel strips, 0.188 with 1 warp and 128, 0.157 with 1 warp and 512) — a view of 1024 pixels is
    // too little work to share: the second warp costs a barrier, a strip counter and its share of per-strip list scans
    if (tiny && c->opt_strip_px <= 0) strip_px = std::max(strip_px, 256);
    const int align = (W & 1) ? 4 : (W & 2) ? 2 : 1;           // strips start on a multiple of 4 pixels
    int SR = align;
    while (SR < 16 && SR * 2 * W <= strip_px) SR *= 2;
    if ((W & (W - 1)) && c->opt_strip_px <= 0) {
        // Width not a power of two: a strip is resolved in groups of 128 consecutive pixels, so the strip height
        // (a multiple of `align`) decides how full the last group is.  Measured on B200: strips of more
        // than ~640 pixels cost occupancy (8-byte key per pixel per warp), fewer than 4 strips per warp cost balance;
        // so take the fullest last group among heights giving <= 640 pixels and enough strips, nearest to 512 pixels
        // on ties, and go up to 1024 pixels only if nothing smaller fills 85 % (210 x 126: 4 rows = 840 pixels).
        // Heights above 2 are multiples of 4: the test tile walks a strip 4 rows at a time.
        const int need = (long long)H * W <= 64 * 64 ? 8 : 16;
        for (int limit = 640; limit <= 1024; limit += 384) {
            double best = -1.0;
            for (int cand = align; cand <= 16; cand += align) {
                const int px = cand * W;
                if (cand > align && (px > limit || (H + cand - 1) / cand < need)) break;
                if (cand > 2 && (cand & 3)) continue;
                const double eff = (double)px / (double)(((px + 127) / 128) * 128);
                if (eff > best) best = eff;
            }
            int best_px = -1;
            for (int cand = align; cand <= 16; cand += align) {
                const int px = cand * W;
                if (cand > align && (px > limit || (H + cand - 1) / cand < need)) break;
                if (cand > 2 && (cand & 3)) continue;
                const double eff = (double)px / (double)(((px + 127) / 128) * 128);
                if (eff >= best - 0.02 && (best_px < 0 || abs(px - 512) < abs(best_px - 512))) { best_px = px; SR = cand; }
            }
            if (best >= 0.85) break;
        }
    }
    pl.SR = SR;
    const int LR = SR >= 4 ? 4 : SR >= 2 ? 2 : 1;              // rows of the test tile (power of two)
    pl.log2LC = LR == 4 ? 3 : LR == 2 ? 4 : 5;
    int log2W = 0;
    while ((1 << log2W) < W) ++log2W;
    pl.log2W = log2W;
    int ng = 0;                                                    // unrolled resolve: NG groups of 128 pixels
    if ((1 << log2W) == W && H % SR == 0 && (SR * W == 128 || SR * W == 256 || SR * W == 512)) ng = SR * W / 128;
    pl.ngr = (ng == 0 && (W & 3) == 0 && (SR * W) % 128 == 0) ? SR * W / 128 : 0;
    pl.magicW = (uint32_t)((0x100000000ull + (unsigned)W - 1) / (unsigned)W);
    const int n_strips = (H + SR - 1) / SR;
    // warps per CTA (= per view): 4; 2 for images of up to 64 x 64 pixels, where twice as many (shorter-lived) CTAs
    // per SM hide the per-view prologue better (32 x 32: 0.230 -> 0.174 ms, 64 x 64: 0.457 -> 0.384 ms; measured slower
    // from 128 x 128 up)
    const int max_warps = tiny ? 1 : (long long)H * W <= 64 * 64 ? (GP_RENDER_WARPS < 2 ? GP_RENDER_WARPS : 2) : GP_RENDER_WARPS;
    int nwarps = n_strips < max_warps ? n_strips : max_warps;
    // List handling (measured on B200): gathering pays when many entries meet a strip — small images
    // (the same list over fewer pixels) or crowded worlds; entry-by-entry is ~1 % faster on the store-bound cases.
    int gather = c->opt_gather;
    if (gather < 0) gather = ((long long)H * W <= 96 * 96 || sc.P >= 400) ? 1 : 0;
    if (sc.P > 65535) gather = 0;                                  // the per-warp overlap list holds 16-bit entry indices
    // shared memory: list stage + row / column tables + per-warp overlap list and key buffer; very wide images
    // get fewer warps per view, and the caller takes the brute-force path if even one warp does not fit
    size_t smem;
    for (;; --nwarps) {
        smem = 48 + (size_t)pl.scap * 64 + (size_t)H * 16 + (size_t)((W + 3) & ~3) * 4 +
               (gather ? (size_t)nwarps * kOverlapCap * sizeof(uint16_t) : 0) + (size_t)nwarps * SR * W * 8;
        if (smem <= 227 * 1024 || nwarps == 1) break;
    }
    // Crowded worlds (the gather mode chosen for P >= 400) are bound by instruction issue, where one more CTA per SM is worth
    // more than a complete list stage: give up staged entries, down to 80, if that lets 8 CTAs of 4 warps fit instead of 7
    // (each CTA costs its shared memory + 1 KB; dense 256 x 256: 30.1 KB -> 27.1 KB, 6.35 -> 6.23 ms).  Store-bound shapes
    // lose with this (sweep 256 x 256 3.97 -> 4.00 ms), 210 x 126 too (4.14 -> 4.24 ms).
    if (c->opt_stage_cap <= 0 && gather && sc.P >= 400 && nwarps == 4 && (smem + 1024) * 8 > 227 * 1024) {
        const size_t budget = 227 * 1024 / 8 - 1024;
        const size_t fixed = smem - (size_t)pl.scap * 64;
        if (fixed + 80 * 64 <= budget) {
            pl.scap = (int)std::min<size_t>((size_t)pl.scap, (budget - fixed) / 64);
            smem = fixed + (size_t)pl.scap * 64;
        }
    }
    pl.ng = ng; pl.nwarps = nwarps; pl.gather = gather; pl.smem = smem;
    return smem <= 227 * 1024;
}

// Launch shape of the raster variant: rows per tile TR (a multiple of the strip alignment, of 4 when > 4 so that the
// 4 x 8 walk of a box stays inside whole row blocks), tiles per view, warps per CTA, shared memory.
struct RasterPlan { int TR, ntiles, nwarps, log2LC, wshift, scap; uint32_t magicW; size_t smem; };
static bool plan_raster(const gp_ctx *c, const SceneConst &sc, int H, int W, RasterPlan &pl) {
    const int align = (W & 1) ? 4 : (W & 2) ? 2 : 1;           // tiles start on a multiple of 4 pixels
    const int tile_px = c->opt_tile_px > 0 ? c->opt_tile_px : 2048;
    int TR = tile_px / W;
    if (TR >= 4) TR &= ~3;
    TR -= TR % align;
    if (TR < align) TR = align;
    if (TR > H) TR = ((H + align - 1) / align) * align;        // one (ragged) tile
    pl.TR = TR;
    pl.ntiles = (H + TR - 1) / TR;
    const int LR = TR >= 4 ? 4 : TR >= 2 ? 2 : 1;
    pl.log2LC = LR == 4 ? 3 : LR == 2 ? 4 : 5;
    int log2W = 0;
    while ((1 << log2W) < W) ++log2W;
    pl.wshift = (1 << log2W) == W ? log2W : -1;
    pl.magicW = (uint32_t)((0x100000000ull + (unsigned)W - 1) / (unsigned)W);
    pl.scap = std::min(sc.P, c->opt_stage_cap > 0 ? c->opt_stage_cap : GP_STAGE_CAP);
    const int groups = (TR * W + 127) / 128;
    pl.nwarps = groups >= 8 ? GP_RASTER_WARPS : groups >= 2 ? 2 : 1;
    pl.smem = 48 + (size_t)pl.scap * 64 + (size_t)TR * 16 + (size_t)((W + 3) & ~3) * 4 + (size_t)TR * W * 8;
    return pl.smem <= 227 * 1024;
}

// The render kernels by template arguments, and their dynamic shared-memory opt-in (raised, never lowered).
typedef void (*RenderFn)(SceneConst, RenderArgs);
#define GP_FNS(ST, SP, GA) {k_render<ST, 0, SP, GA>, k_render<ST, 1, SP, GA>, k_render<ST, 2, SP, GA>, k_render<ST, 4, SP, GA>}
static const RenderFn kRenderFns[2][2][2][4] = {      // [gather][spheres][stats][ng index]
    {{GP_FNS(false, false, false), GP_FNS(true, false, false)}, {GP_FNS(false, true, false), GP_FNS(true, true, false)}},
    {{GP_FNS(false, false, true), GP_FNS(true, false, true)}, {GP_FNS(false, true, true), GP_FNS(true, true, true)}}};
#undef GP_FNS
static const RenderFn kRasterFns[2][2] = {{k_raster<false, false>, k_raster<true, false>},
                                          {k_raster<false, true>, k_raster<true, true>}};     // [spheres][stats]
static int set_render_smem(gp_ctx *c, size_t smem) {
    if (smem <= c->render_smem_set) return GP_OK;
    for (int ga = 0; ga < 2; ++ga)
        for (int f = 0; f < 2; ++f)
            for (int st = 0; st < 2; ++st)
                for (int g = 0; g < 4; ++g)
                    CK(cudaFuncSetAttribute(kRenderFns[ga][f][st][g], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    c->render_smem_set = smem;
    return GP_OK;
}
static int set_raster_smem(gp_ctx *c, size_t smem) {
    if (smem <= c->raster_smem_set) return GP_OK;
    for (int f = 0; f < 2; ++f)
        for (int st = 0; st < 2; ++st)
            CK(cudaFuncSetAttribute(kRasterFns[f][st], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    c->raster_smem_set = smem;
    return GP_OK;
}

// Enqueue cull + render (or the brute-force kernel) for a world range into DEVICE planes.
static int render_device(gp_ctx *c, int world_begin, int n_worlds, int H, int W, float fov_rad,
                         uint8_t *d_class, int32_t *d_instance, float *d_depth, uint8_t *d_rgb,
                         cudaStream_t stream) {
    // Spheres are drawn iff the uploaded scene held one or gp_statics_update has run since (its records are device
    // memory the host never sees), unless GP_OPT_SPHERES says otherwise; when off, sphere records are skipped by
    // every path alike (cull and brute force), so the result stays well defined.
    const bool spheres = c->opt_spheres >= 0 ? c->opt_spheres != 0 : (c->has_spheres || c->statics_touched);
    SceneConst sc = c->sc;
    sc.spheres = spheres ? 1 : 0;
    c->last_H = H; c->last_W = W;
    const float th = (float)tan(0.5 * (double)fov_rad);          // C2, host side
    const float tv = th * ((float)H / (float)W);
    const size_t views = (size_t)n_worlds * sc.A * sc.C;
    if (views > 0x7fffffffull) return GP_ERR_ARG;
    unsigned long long *stats = c->opt_stats ? c->d_stats : nullptr;
    if (stats) CK(cudaMemsetAsync(stats, 0, 2 * sizeof(unsigned long long), stream));

    // fast path: every view (H*W pixels) must start 16-byte aligned in the 32-bit planes, and one warp's strip
    // must fit shared memory (it does not for e.g. 4096 x 4094: odd widths force 2- or 4-row strips)
    RenderPlan pl{};
    RasterPlan rp{};
    int variant = c->opt_variant;
    if (variant < 0) variant = GP_VARIANT_RAY;
    const bool size_ok = W >= 4 && !(((long long)H * W) & 3);
    if (variant == GP_VARIANT_RASTER && !(size_ok && plan_raster(c, sc, H, W, rp))) variant = GP_VARIANT_RAY;
    const bool fast_ok = size_ok && (variant == GP_VARIANT_RASTER || plan_render(c, sc, H, W, pl));
    if (c->opt_path == GP_PATH_BRUTE || !fast_ok) {
        const int HW = H * W;
        dim3 grid((unsigned)views, (unsigned)std::min((HW + 255) / 256, 65535));
        {
            LaunchTimer lt(c, GP_KERNEL_BRUTE, stream);
            k_render_brute<<<grid, 256, 0, stream>>>(sc, c->d_prims, c->d_pitch, world_begin, H, W, th, tv,
                                                      d_class, d_instance, d_depth, d_rgb, nullptr);
        }
        c->launches += 1;
        CK(cudaGetLastError());
        return GP_OK;
    }
    int rc = ensure_scratch(c, views);
    if (rc != GP_OK) return rc;
    // Capped lists: the overflow flags are cleared here, BEFORE the fork below, so that the culls on the side stream (which
    // wait only for the fork event) are ordered behind the clear; issued later on `stream` it could wipe a flag a side-stream
    // cull had already set, and that view would keep its background-only image
    const bool capped = c->scratch_cap < sc.P;                         // lists may overflow: flag + brute-force repair pass
    if (capped) CK(cudaMemsetAsync(c->d_ovf, 0, views, stream));

    // ---- pipeline over world chunks: the cull of chunk i + 1 runs on a library-owned high-priority stream while chunk i
    // renders on the caller's stream (the cull is bound by instruction issue and latency, the render by HBM stores,
    // so they overlap well; serially the cull costs 8 % of the paper-scale step).  Fork / join by events, capturable in
    // a CUDA graph.  Every chunk has its own slice of the per-view scratch, so culls may run arbitrarily far ahead.
    const int vpw = sc.A * sc.C;                                       // views per world
    int n_chunks = c->opt_pipeline;                                    // default 1: measured slower than serial
    n_chunks = std::min(n_chunks, n_worlds);
    if (stats || n_chunks < 1) n_chunks = 1;
    const int wpc = (n_worlds + n_chunks - 1) / n_chunks;              // worlds per chunk
    n_chunks = (n_worlds + wpc - 1) / wpc;
    cudaStream_t cull_stream = stream;
    if (n_chunks > 1) {
        if (!c->aux_stream) {
            int lo = 0, hi = 0;
            CK(cudaDeviceGetStreamPriorityRange(&lo, &hi));
            CK(cudaStreamCreateWithPriority(&c->aux_stream, cudaStreamNonBlocking, hi));
        }
        while ((int)c->pipe_ev.size() < n_chunks + 1) {
            cudaEvent_t e;
            CK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            c->pipe_ev.push_back(e);
        }
        cull_stream = c->aux_stream;
        CK(cudaEventRecord(c->pipe_ev[n_chunks], stream));             // fork: the culls see everything enqueued so far
        CK(cudaStreamWaitEvent(cull_stream, c->pipe_ev[n_chunks], 0));
    }
    const int gpw = (vpw + kCullWarps - 1) / kCullWarps;               // cull CTAs per world
    CullArgs cargs{};
    cargs.prims = c->d_prims; cargs.pitch = c->d_pitch; cargs.groups_per_world = gpw; cargs.H = H; cargs.W = W;
    cargs.th = th; cargs.tv = tv;
    cargs.sth = sqrtf(fmaf(th, th, 1.0f)) * 1.0001f; cargs.stv = sqrtf(fmaf(tv, tv, 1.0f)) * 1.0001f;
    cargs.msc = 2.0f + th + tv;
    cargs.inv_th = 1.0f / th; cargs.inv_tv = 1.0f / tv; cargs.halfW = 0.5f * (float)W; cargs.halfH = 0.5f * (float)H;
    cargs.far_lim = sc.t_max * (1.0f + 1e-6f);
    cargs.cap = c->scratch_cap; cargs.stats = stats;
    auto launch_cull = [&](int ci, cudaStream_t st) -> int {
        const int w0 = ci * wpc, nw = std::min(wpc, n_worlds - w0);
        const size_t v0 = (size_t)w0 * vpw;
        CullArgs ca = cargs;
        ca.world_begin = world_begin + w0;
        ca.hdr = c->d_hdr + v0; ca.geo = c->d_geo + v0 * c->scratch_cap; ca.aux = c->d_aux + v0 * c->scratch_cap;
        ca.ovf = capped ? c->d_ovf + v0 : nullptr;
        {
            LaunchTimer lt(c, GP_KERNEL_CULL, st);
#if GP_PDL
            if (st == stream) {        // behind whatever the caller enqueued last (usually the pose update)
                cudaLaunchConfig_t cfg = {};
                cfg.gridDim = dim3((unsigned)((size_t)nw * gpw)); cfg.blockDim = dim3(kCullWarps * 32); cfg.stream = st;
                cudaLaunchAttribute at[1];
                at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
                at[0].val.programmaticStreamSerializationAllowed = 1;
                cfg.attrs = at; cfg.numAttrs = 1;
                CK(cudaLaunchKernelEx(&cfg, capped ? k_cull<true> : k_cull<false>, sc, ca));
            } else
#endif
            if (capped) k_cull<true><<<(unsigned)((size_t)nw * gpw), kCullWarps * 32, 0, st>>>(sc, ca);
            else k_cull<false><<<(unsigned)((size_t)nw * gpw), kCullWarps * 32, 0, st>>>(sc, ca);
        }
        c->launches += 1;
        CK(cudaGetLastError());
        return GP_OK;
    };

    RenderArgs ra{};
    ra.meta = c->d_meta;
    ra.two_over_H = 2.0f / (float)H; ra.two_over_W = 2.0f / (float)W;
    ra.cap = c->scratch_cap; ra.H = H; ra.W = W; ra.th = th; ra.tv = tv; ra.stats = stats;
    RenderFn fn = nullptr;
    unsigned ctas_per_view = 1, block = 0;
    size_t smem = 0;
    if (variant == GP_VARIANT_RASTER) {
        ra.scap = rp.scap; ra.SR = rp.TR; ra.log2LC = rp.log2LC; ra.log2W = rp.wshift; ra.magicW = rp.magicW; ra.ntiles = rp.ntiles;
        rc = set_raster_smem(c, rp.smem);
        if (rc != GP_OK) return rc;
        if (views * (size_t)rp.ntiles > 0x7fffffffull) return GP_ERR_ARG;
        fn = kRasterFns[spheres ? 1 : 0][stats ? 1 : 0];
        ctas_per_view = (unsigned)rp.ntiles; block = (unsigned)rp.nwarps * 32; smem = rp.smem;
    } else {
        ra.scap = pl.scap; ra.SR = pl.SR; ra.log2LC = pl.log2LC; ra.log2W = pl.log2W; ra.ngr = pl.ngr; ra.magicW = pl.magicW;
        ra.n_strips = (H + pl.SR - 1) / pl.SR;
        ra.magicSR = (uint32_t)((0x100000000ull + (unsigned)pl.SR - 1) / (unsigned)pl.SR);
        rc = set_render_smem(c, pl.smem);
        if (rc != GP_OK) return rc;
        fn = kRenderFns[pl.gather][spheres ? 1 : 0][stats ? 1 : 0][pl.ng == 4 ? 3 : pl.ng];
        block = (unsigned)pl.nwarps * 32; smem = pl.smem;
    }
    {   // view / vpw for view < 2^31: (view * ceil(2^(31 + L) / vpw)) >> (31 + L), L = ceil(log2 vpw) (round-up method)
        int L = 0;
        while ((1ll << L) < vpw) ++L;
        ra.shift_vpw = 31 + L;
        ra.magic_vpw = (uint32_t)(((1ull << (31 + L)) + (unsigned)vpw - 1) / (unsigned)vpw);
    }
    const size_t HW = (size_t)H * W;
    rc = launch_cull(0, stream);                                       // chunk 0: nothing to overlap with yet
    if (rc != GP_OK) return rc;
    for (int ci = 1; ci < n_chunks; ++ci) {                            // the other culls run ahead on the side stream
        rc = launch_cull(ci, cull_stream);
        if (rc != GP_OK) return rc;
        CK(cudaEventRecord(c->pipe_ev[ci], cull_stream));
    }
    for (int ci = 0; ci < n_chunks; ++ci) {
        const int w0 = ci * wpc, nw = std::min(wpc, n_worlds - w0);
        const size_t v0 = (size_t)w0 * vpw, nv = (size_t)nw * vpw;
        if (ci > 0) CK(cudaStreamWaitEvent(stream, c->pipe_ev[ci], 0));  // join (the last one joins the side stream for good)
        ra.hdr = c->d_hdr + v0; ra.geo = c->d_geo + v0 * c->scratch_cap; ra.aux = c->d_aux + v0 * c->scratch_cap;
        ra.world_begin = world_begin + w0;
        ra.o_cls = d_class + v0 * HW; ra.o_inst = d_instance + v0 * HW; ra.o_depth = d_depth + v0 * HW;
        ra.o_rgb = d_rgb ? d_rgb + v0 * 3 * HW : nullptr;
        {
            LaunchTimer lt(c, GP_KERNEL_RENDER, stream);
#if GP_PDL
            if (variant == GP_VARIANT_RAY && n_chunks == 1) {
                // programmatic dependent launch on the cull enqueued just before: the render CTAs may become resident and
                // run their view-independent prologue while the cull's last CTAs finish (griddepcontrol.wait in k_render)
                cudaLaunchConfig_t cfg = {};
                cfg.gridDim = dim3((unsigned)(nv * ctas_per_view)); cfg.blockDim = dim3(block);
                cfg.dynamicSmemBytes = smem; cfg.stream = stream;
                cudaLaunchAttribute at[1];
                at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
                at[0].val.programmaticStreamSerializationAllowed = 1;
                cfg.attrs = at; cfg.numAttrs = 1;
                CK(cudaLaunchKernelEx(&cfg, fn, sc, ra));
            } else
#endif
            fn<<<dim3((unsigned)(nv * ctas_per_view)), dim3(block), smem, stream>>>(sc, ra);
        }
        c->launches += 1;
        CK(cudaGetLastError());
    }
    if (capped) {
        // repair pass: the views whose list overflowed the cap (the render pass drew only the background for them) are
        // rendered by the brute-force kernel, one CTA per flagged view; the CTAs of all other views exit at once
        {
            LaunchTimer lt(c, GP_KERNEL_BRUTE, stream);
            k_render_brute<<<dim3((unsigned)views, 1), 256, 0, stream>>>(sc, c->d_prims, c->d_pitch, world_begin, H, W, th, tv,
                                                                           d_class, d_instance, d_depth, d_rgb, c->d_ovf);
        }
        c->launches += 1;
        CK(cudaGetLastError());
    }
    return GP_OK;
}

extern "C" int gp_reserve(gp_ctx *c, int n_worlds, int H, int W) {
    if (!c) return GP_ERR_ARG;
    if (!c->have_scene) return GP_ERR_STATE;
    if (H < 1 || W < 1 || H > 4096 || W > 4096 || n_worlds < 1) return GP_ERR_ARG;
    if (n_worlds > c->sc.Wn) return GP_ERR_RANGE;
    GP_ON_DEVICE(c);
    const size_t views = (size_t)n_worlds * c->sc.A * c->sc.C;
    if (views > 0x7fffffffull) return GP_ERR_ARG;
    int rc = ensure_scratch(c, views);
    if (rc != GP_OK) return rc;
    if (W >= 4 && !(((long long)H * W) & 3)) {
        RenderPlan pl{}; RasterPlan rp{};
        if (plan_render(c, c->sc, H, W, pl) && (rc = set_render_smem(c, pl.smem)) != GP_OK) return rc;
        if (plan_raster(c, c->sc, H, W, rp) && (rc = set_raster_smem(c, rp.smem)) != GP_OK) return rc;
    }
    return GP_OK;
}

extern "C" int gp_render_batch(gp_ctx *c, int world_begin, int n_worlds, int agents, int H, int W,
                               float fov_rad, uint8_t *d_class, int32_t *d_instance, float *d_depth,
                               uint8_t *d_rgb, void *stream_) {
    int rc = check_render_args(c, world_begin, n_worlds, agents, H, W, fov_rad);
    if (rc != GP_OK) return rc;
    if (!d_class || !d_instance || !d_depth) return GP_ERR_ARG;
    if (!aligned16(d_class) || !aligned16(d_instance) || !aligned16(d_depth) || !aligned16(d_rgb)) return GP_ERR_ALIGN;
    GP_ON_DEVICE(c);
    return render_device(c, world_begin, n_worlds, H, W, fov_rad, d_class, d_instance, d_depth, d_rgb,
                         static_cast<cudaStream_t>(stream_));
}

extern "C" int gp_render_batch_host(gp_ctx *c, const float *h_pose, int world_begin, int n_worlds, int agents,
                                    int H, int W, float fov_rad, uint8_t *h_class, int32_t *h_instance,
                                    float *h_depth, uint8_t *h_rgb, void *stream_) {
    int rc = check_render_args(c, world_begin, n_worlds, agents, H, W, fov_rad);
    if (rc != GP_OK) return rc;
    if (!h_class && !h_instance && !h_depth && !h_rgb) return GP_ERR_ARG;
    GP_ON_DEVICE(c);
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const SceneConst &sc = c->sc;
    const size_t HW = (size_t)H * W, A = (size_t)sc.A * sc.C;      // A: views per world here
    const size_t bpv = HW * 12;                                   // staged bytes per view (all planes are rendered)
    // chunk: <= 512 MiB of planes per staging buffer, at least one world
    size_t wc = (512ull << 20) / (bpv * A);
    if (wc < 1) wc = 1;
    if (wc > (size_t)n_worlds) wc = n_worlds;
    const size_t plane = (wc * A * HW + 255) & ~(size_t)255;       // staging plane stride in elements
    const size_t need = plane * 12;
    if (!c->copy_stream) {
        CK(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CK(cudaEventCreateWithFlags(&c->ev_render[i], cudaEventDisableTiming));
            CK(cudaEventCreateWithFlags(&c->ev_copy[i], cudaEventDisableTiming));
        }
    }
    if (c->d_out_bytes < need) {
        CK(cudaDeviceSynchronize());
        for (int i = 0; i < 2; ++i) { cudaFree(c->d_out[i]); c->d_out[i] = nullptr; }
        c->d_out_bytes = 0;
        for (int i = 0; i < 2; ++i)
            if (cudaMalloc(&c->d_out[i], need) != cudaSuccess) { cudaGetLastError(); return GP_ERR_NOMEM; }
        c->d_out_bytes = need;
    }
    if (h_pose) {
        CK(cudaMemcpyAsync(c->d_pose, h_pose, (size_t)sc.Wn * sc.A * 4 * sizeof(float), cudaMemcpyHostToDevice, stream));
        rc = gp_agents_update(c, c->d_pose, stream);
        if (rc != GP_OK) return rc;
    }
    int buf = 0;
    for (size_t w0 = 0; w0 < (size_t)n_worlds; w0 += wc, buf ^= 1) {
        const size_t nw = std::min(wc, (size_t)n_worlds - w0), nv = nw * A;
        unsigned char *base = c->d_out[buf];
        uint8_t *dc = base; int32_t *di = reinterpret_cast<int32_t *>(base + plane);
        float *dd = reinterpret_cast<float *>(base + plane * 5);
        uint8_t *dr = h_rgb ? base + plane * 9 : nullptr;           // the rgb plane is not even rendered when unwanted
        CK(cudaStreamWaitEvent(stream, c->ev_copy[buf], 0));      // staging buffer free again
        rc = render_device(c, world_begin + (int)w0, (int)nw, H, W, fov_rad, dc, di, dd, dr, stream);
        if (rc != GP_OK) return rc;
        CK(cudaEventRecord(c->ev_render[buf], stream));
        CK(cudaStreamWaitEvent(c->copy_stream, c->ev_render[buf], 0));
        const size_t v0 = w0 * A;
        if (h_class) CK(cudaMemcpyAsync(h_class + v0 * HW, dc, nv * HW, cudaMemcpyDeviceToHost, c->copy_stream));
        if (h_instance) CK(cudaMemcpyAsync(h_instance + v0 * HW, di, nv * HW * 4, cudaMemcpyDeviceToHost, c->copy_stream));
        if (h_depth) CK(cudaMemcpyAsync(h_depth + v0 * HW, dd, nv * HW * 4, cudaMemcpyDeviceToHost, c->copy_stream));
        if (h_rgb) CK(cudaMemcpyAsync(h_rgb + v0 * HW * 3, dr, nv * HW * 3, cudaMemcpyDeviceToHost, c->copy_stream));
        CK(cudaEventRecord(c->ev_copy[buf], c->copy_stream));
    }
    CK(cudaStreamSynchronize(c->copy_stream));
    CK(cudaStreamSynchronize(stream));
    return GP_OK;
}

extern "C" int gp_probe(gp_ctx *c, int kind, size_t n_pixels, int iters, uint8_t *d_class, int32_t *d_instance,
                        float *d_depth, uint8_t *d_rgb, void *stream_, double *best, double *median) {
    if (!c || !best || iters < 1 || iters > 1000) return GP_ERR_ARG;
    GP_ON_DEVICE(c);
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    { cudaError_t e = cudaEventCreate(&e1); if (e != cudaSuccess) { cudaEventDestroy(e0); return cuda_fail(e, "cudaEventCreate"); } }
    unsigned long long *d_probe = c->d_stats + 2;               // the probes' own words: the GP_OPT_STATS counters stay intact
    const unsigned probe_grid = (unsigned)c->n_sms * 8;
    std::vector<double> rate;
    int rc = GP_OK;
    for (int it = 0; it < iters + 1 && rc == GP_OK; ++it) {                 // the first launch is a warm-up
        cudaEventRecord(e0, stream);
        double units = 0.0;
        if (kind == GP_PROBE_STORE) {
            if (!d_class || !d_instance || !d_depth || !d_rgb || n_pixels < 128 || (n_pixels & 127)) { rc = GP_ERR_ARG; break; }
            if (!aligned16(d_class) || !aligned16(d_instance) || !aligned16(d_depth) || !aligned16(d_rgb)) { rc = GP_ERR_ALIGN; break; }
            const size_t groups = n_pixels / 128;
            k_probe_store<<<(unsigned)((groups + 15) / 16), 128, 0, stream>>>(groups, d_class, d_instance, d_depth, d_rgb,
                                                                                n_pixels, 0x01010101u * (uint32_t)(it & 3));
            units = (double)n_pixels * 12.0 / 1e9;                              // GB
        } else if (kind == GP_PROBE_STORE_VIEW) {
            const size_t HW = (size_t)c->last_H * c->last_W;
            if (HW == 0) { rc = GP_ERR_STATE; break; }
            if (!d_class || !d_instance || !d_depth || !d_rgb || (HW & 127) || n_pixels < HW || n_pixels % HW ||
                n_pixels / HW > 0x7fffffffull) { rc = GP_ERR_ARG; break; }
            if (!aligned16(d_class) || !aligned16(d_instance) || !aligned16(d_depth) || !aligned16(d_rgb)) { rc = GP_ERR_ALIGN; break; }
            k_probe_store_view<<<(unsigned)(n_pixels / HW), 128, 0, stream>>>((int)(HW / 128), d_class, d_instance, d_depth, d_rgb,
                                                                              0x01010101u * (uint32_t)(it & 3));
            units = (double)n_pixels * 12.0 / 1e9;                              // GB
        } else if (kind == GP_PROBE_FMA) {
            const int reps = 4096;
            k_probe_fma<<<probe_grid, 256, 0, stream>>>(reps, 1.0f + (float)it, reinterpret_cast<float *>(d_probe));
            units = 2.0 * (double)probe_grid * 256 * (double)reps * 16 * 8 / 1e12;   // TFLOP
        } else if (kind == GP_PROBE_RCP) {
            if (it == 0) {                                                                          // count over all launches
                cudaError_t e = cudaMemsetAsync(d_probe, 0, sizeof(unsigned long long), stream);
                if (e != cudaSuccess) { rc = cuda_fail(e, "cudaMemsetAsync(probe)"); break; }
            }
            k_probe_rcp<<<probe_grid, 256, 0, stream>>>(d_probe);
            units = 0.0;
        } else { rc = GP_ERR_ARG; break; }
        c->launches += 1;
        cudaEventRecord(e1, stream);
        if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) { rc = cuda_fail(cudaGetLastError(), "gp_probe"); break; }
        float ms = 0.0f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (it > 0) rate.push_back(units / (ms * 1e-3));
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (rc != GP_OK) return rc;
    if (kind == GP_PROBE_RCP) {                                                 // result = mismatching bit patterns
        unsigned long long bad = 0;
        CK(cudaMemcpy(&bad, d_probe, sizeof bad, cudaMemcpyDeviceToHost));
        CK(cudaMemset(d_probe, 0, sizeof bad));
        *best = (double)bad;
        if (median) *median = (double)bad;
        return GP_OK;
    }
    std::sort(rate.begin(), rate.end());
    *best = rate.back();
    if (median) *median = rate[rate.size() / 2];
    return GP_OK;
}

extern "C" int gp_stats(gp_ctx *c, uint64_t *executed_tests, uint64_t *listed_pairs) {
    if (!c) return GP_ERR_ARG;
    unsigned long long h[2];
    GP_ON_DEVICE(c);
    CK(cudaDeviceSynchronize());
    CK(cudaMemcpy(h, c->d_stats, sizeof h, cudaMemcpyDeviceToHost));
    if (executed_tests) *executed_tests = h[0];
    if (listed_pairs) *listed_pairs = h[1];
    return GP_OK;
}

extern "C" int gp_kernel_time(gp_ctx *c, int kernel, double *total_ms, uint64_t *launches) {
    if (!c || !total_ms || !launches) return GP_ERR_ARG;
    GP_ON_DEVICE(c);
    CK(cudaDeviceSynchronize());
    double ms = 0.0; uint64_t n = 0;
    std::vector<gp_ctx::Timed> keep;
    for (const auto &t : c->timed) {
        if (t.kernel != kernel) { keep.push_back(t); continue; }
        float x = 0.0f;
        if (cudaEventElapsedTime(&x, t.a, t.b) == cudaSuccess) { ms += x; ++n; }
        c->ev_pool.push_back(t.a); c->ev_pool.push_back(t.b);
    }
    c->timed.swap(keep);
    *total_ms = ms; *launches = n;
    return GP_OK;
}

extern "C" int gp_launch_count(gp_ctx *c, uint64_t *launches) {
    if (!c || !launches) return GP_ERR_ARG;
    *launches = c->launches;
    return GP_OK;
}

// ---- gp_render_static: the render step for callers that must not allocate (include/gp.h) ---------------------------
//
// Some processes cannot let this library call cudaMalloc: the training framework already owns all of HBM, or the loop
// cannot afford the device-wide stall of an allocation, or device memory is budgeted to the byte.  For them the
// intermediates of cull + render live in the fixed array below instead of a gp_ctx.  The array is part of the library
// image: every GPU of a process that loads libgp.so carries its kStBytes from load to exit.  Sections (each starts on a
// multiple of 256 bytes):
namespace {
constexpr size_t kStHdr = 0;                                                               // ViewHdr  [MAX_VIEWS]
constexpr size_t kStPitch = kStHdr + (size_t)GP_STATIC_MAX_VIEWS * sizeof(ViewHdr);       // float2   [MAX_VIEWS]   (pitch 0)
constexpr size_t kStMeta = kStPitch + (size_t)GP_STATIC_MAX_VIEWS * sizeof(float2);       // PrimMeta [MAX_PRIMS]
constexpr size_t kStGeo = kStMeta + (size_t)GP_STATIC_MAX_PRIMS * sizeof(PrimMeta);       // EntryGeo [MAX_ENTRIES]
constexpr size_t kStAux = kStGeo + (size_t)GP_STATIC_MAX_ENTRIES * sizeof(EntryGeo);      // EntryAux [MAX_ENTRIES]
constexpr size_t kStBytes = kStAux + (size_t)GP_STATIC_MAX_ENTRIES * sizeof(EntryAux);
static_assert(kStPitch % 256 == 0 && kStMeta % 256 == 0 && kStGeo % 256 == 0 && kStAux % 256 == 0, "section alignment");
static_assert(kStBytes == 9535488, "include/gp.h states this size");
constexpr int kStMaxDevices = 64;
}  // namespace

static __device__ __align__(256) unsigned char g_static_scratch[kStBytes];

// In host code `g_static_scratch` is only a handle for the runtime, not an address a kernel could use: the address on
// each device comes from cudaGetSymbolAddress, asked once per device with that device current, and is kept here.
static std::mutex g_static_mu;
static unsigned char *g_static_base[kStMaxDevices];

static int static_scratch_base(int dev, unsigned char **base) {      // the caller has made `dev` current
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_base[dev]) {
        int major = 0;
        CK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        if (major != 10) return GP_ERR_ARCH;
        unsigned char *p = nullptr;
        CK(cudaGetSymbolAddress(reinterpret_cast<void **>(&p), g_static_scratch));
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255u)) return cuda_fail(cudaErrorInvalidSymbol, "cudaGetSymbolAddress(g_static_scratch)");
        g_static_base[dev] = p;
    }
    *base = g_static_base[dev];
    return GP_OK;
}

extern "C" int gp_render_static(int cuda_device, const gp_scene_desc *d, const gp_prim *d_prims, const float *d_pitch_cs,
                                int H, int W, float fov_rad, uint8_t *d_class, int32_t *d_instance, float *d_depth,
                                uint8_t *d_rgb, void *stream_) {
    if (!d || !d_prims || !d_class || !d_instance || !d_depth) return GP_ERR_ARG;
    if (cuda_device < 0 || cuda_device >= kStMaxDevices) return GP_ERR_ARG;
    if (d->n_worlds < 1 || d->agents_per_world < 1 || d->quads_per_world < 0) return GP_ERR_ARG;
    if (!(d->cam_height > 0.0f) || !(d->t_max > 0.0f) || !(d->ambient >= 0.0f && d->ambient <= 1.0f)) return GP_ERR_ARG;
    if (H < 1 || W < 4 || H > 4096 || W > 4096 || (((long long)H * W) & 3)) return GP_ERR_ARG;
    if (!(fov_rad > 0.0f && fov_rad < 3.1415f)) return GP_ERR_ARG;
    if (!aligned16(d_prims) || !aligned16(d_class) || !aligned16(d_instance) || !aligned16(d_depth) || !aligned16(d_rgb) ||
        (reinterpret_cast<uintptr_t>(d_pitch_cs) & 7u)) return GP_ERR_ALIGN;
    // the fixed scratch bounds the scene: refuse anything larger before touching the device
    const long long P = (long long)d->agents_per_world + d->quads_per_world;
    const long long views = (long long)d->n_worlds * d->agents_per_world;
    if (views > GP_STATIC_MAX_VIEWS || (long long)d->n_worlds * P > GP_STATIC_MAX_PRIMS || views * P > GP_STATIC_MAX_ENTRIES)
        return GP_ERR_LIMIT;

    gp_ctx plan_opts;                      // launch-shape rules of the ordinary path with every option at its default
    plan_opts.device = cuda_device;        // (host object only: it owns no device memory and is never passed to a kernel)
    GP_ON_DEVICE(&plan_opts);
    unsigned char *base = nullptr;
    int rc = static_scratch_base(cuda_device, &base);
    if (rc != GP_OK) return rc;
    ViewHdr *s_hdr = reinterpret_cast<ViewHdr *>(base + kStHdr);
    float2 *s_pitch = reinterpret_cast<float2 *>(base + kStPitch);
    PrimMeta *s_meta = reinterpret_cast<PrimMeta *>(base + kStMeta);
    EntryGeo *s_geo = reinterpret_cast<EntryGeo *>(base + kStGeo);
    EntryAux *s_aux = reinterpret_cast<EntryAux *>(base + kStAux);

    SceneConst sc{};
    sc.Wn = d->n_worlds; sc.A = d->agents_per_world; sc.Q = d->quads_per_world; sc.P = (int)P;
    sc.C = 1; sc.rig[0] = make_float4(1.0f, 0.0f, 1.0f, 0.0f);            // the default rig: one front-centre camera
    sc.spheres = 1;                                                       // the records are never seen by the host
    sc.cam_h = d->cam_height; sc.t_max = d->t_max;
    sc.Lx = d->light[0]; sc.Ly = d->light[1]; sc.Lz = d->light[2]; sc.ambient = d->ambient;
    for (int k = 0; k < 8; ++k)
        sc.pal[k] = (uint32_t)d->palette[k][0] | ((uint32_t)d->palette[k][1] << 8) | ((uint32_t)d->palette[k][2] << 16);
    RenderPlan pl{};
    if (!plan_render(&plan_opts, sc, H, W, pl)) return GP_ERR_ARG;       // not even one warp's strip fits shared memory
    const RenderFn fn = kRenderFns[pl.gather][1][0][pl.ng == 4 ? 3 : pl.ng];
    // Permit the kernel the largest dynamic shared memory there is, on every call: contexts on this device raise and lower
    // the same attribute for their own needs, and the maximum satisfies all of them
    CK(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));

    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const float th = (float)tan(0.5 * (double)fov_rad);                   // C2, host side
    const float tv = th * ((float)H / (float)W);
    const int vpw = sc.A;
    // The array still holds the previous call's headers and lists.  Each header read below is rewritten by this call's
    // cull first; clearing them costs 16 bytes per view and rules out a stale list length whatever else goes wrong.
    CK(cudaMemsetAsync(s_hdr, 0, (size_t)views * sizeof(ViewHdr), stream));
    k_prim_meta<<<(unsigned)(((size_t)sc.Wn * sc.P + 255) / 256), 256, 0, stream>>>(sc, d_prims, s_meta);
    if (!d_pitch_cs) k_fill_pitch<<<(unsigned)((views + 255) / 256), 256, 0, stream>>>(s_pitch, (size_t)views);
    CK(cudaGetLastError());

    const int gpw = (vpw + kCullWarps - 1) / kCullWarps;
    CullArgs ca{};
    ca.prims = d_prims; ca.pitch = d_pitch_cs ? reinterpret_cast<const float2 *>(d_pitch_cs) : s_pitch;
    ca.world_begin = 0; ca.groups_per_world = gpw; ca.H = H; ca.W = W; ca.th = th; ca.tv = tv;
    ca.sth = sqrtf(fmaf(th, th, 1.0f)) * 1.0001f; ca.stv = sqrtf(fmaf(tv, tv, 1.0f)) * 1.0001f;
    ca.msc = 2.0f + th + tv;
    ca.inv_th = 1.0f / th; ca.inv_tv = 1.0f / tv; ca.halfW = 0.5f * (float)W; ca.halfH = 0.5f * (float)H;
    ca.far_lim = sc.t_max * (1.0f + 1e-6f);
    ca.hdr = s_hdr; ca.geo = s_geo; ca.aux = s_aux; ca.cap = sc.P;        // a list can hold the whole world: no overflow
    ca.ovf = nullptr; ca.stats = nullptr;
    k_cull<false><<<(unsigned)((size_t)sc.Wn * gpw), kCullWarps * 32, 0, stream>>>(sc, ca);
    CK(cudaGetLastError());

    RenderArgs ra{};
    ra.hdr = s_hdr; ra.geo = s_geo; ra.aux = s_aux; ra.meta = s_meta;
    ra.cap = sc.P; ra.scap = pl.scap; ra.world_begin = 0; ra.H = H; ra.W = W; ra.th = th; ra.tv = tv;
    ra.SR = pl.SR; ra.log2LC = pl.log2LC; ra.log2W = pl.log2W; ra.ngr = pl.ngr; ra.magicW = pl.magicW;
    ra.o_cls = d_class; ra.o_inst = d_instance; ra.o_depth = d_depth; ra.o_rgb = d_rgb; ra.stats = nullptr;
    ra.n_strips = (H + pl.SR - 1) / pl.SR;
    ra.magicSR = (uint32_t)((0x100000000ull + (unsigned)pl.SR - 1) / (unsigned)pl.SR);
    ra.two_over_H = 2.0f / (float)H; ra.two_over_W = 2.0f / (float)W;
    {
        int L = 0;
        while ((1ll << L) < vpw) ++L;
        ra.shift_vpw = 31 + L;
        ra.magic_vpw = (uint32_t)(((1ull << (31 + L)) + (unsigned)vpw - 1) / (unsigned)vpw);
    }
    fn<<<dim3((unsigned)views), dim3((unsigned)pl.nwarps * 32), pl.smem, stream>>>(sc, ra);
    CK(cudaGetLastError());
    return GP_OK;
}
