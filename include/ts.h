/* ts.h -- C ABI of the B200-native batched tactile readout (after Tactile Genesis,
 * arxiv/paper_2606_22332; "P:NNN" = line NNN of the paper text, App. A = P:172-359).
 *
 * One context (ts_ctx) serves E environments x T taxel slots on ONE CUDA device.  Each
 * ts_step() runs, for every (environment, taxel):
 *   Eq. 1      q_j = p_L + R_L x_j,  a_j = R_L n_j
 *   Eq. 2      d_j = max_g [R_j - phi_g(q_j)]_+ , normal m_j = grad phi_g*
 *   Eq. 3      Schmitt-trigger contact bit
 *   Eq. 4-9  kinematic force / torque (+ Coulomb cap, D2)
 *   Eq. 18-21, 23  elastomer marker dilation
 *   bounded SDF march along a_j (D1; output form of Eq. 12)
 *   App. A.8 noise: [gain (Eq. 27)] -> hysteresis (Eq. 29-30) -> crosstalk (Eq. 31) ->
 *                        [bias + white noise +] random-walk drift (Eq. 25) [-> quantize (Eq. 25)] ->
 *                        dead taxels (Eq. 28); bracketed knobs are off by default
 * All device work is hand-written CUDA for sm_100a; there is no CPU fallback.
 *
 * Conventions: SI units; quaternions (w,x,y,z), used as given (never renormalised); each
 * environment has its own world frame; force/torque and marker outputs are expressed in the
 * sensor-link frame.  All arrays are dense, row-major, fp32 unless stated.
 *
 * Threading: calls on one ctx are not thread-safe.  Streams: every device operation of
 * ts_set_geometry / ts_step / ts_reset is enqueued on the caller's stream (a cudaStream_t
 * passed as void*; NULL = the legacy default stream); none of them synchronises except where
 * stated.  The ctx keeps state between calls (Schmitt bits, hysteresis, drift, counters, the
 * frames of the step in flight), so successive calls on one ctx must be ordered: use ONE stream,
 * or order the streams yourself with events; the library does not check this.
 * Programmatic dependent launch: within a step the readout kernel is launched as a programmatic dependent of the
 * pose kernel, and the pose kernel of the NEXT ts_step as a dependent of this step's readout kernel, so when ts_step
 * calls are enqueued back to back on one stream the launch latencies and block ramp-up are hidden behind the kernel in
 * front.  The pose kernel still waits, on the device, for everything enqueued in front of it (the caller's kernels that
 * produce the next poses included) to complete and become visible before it reads anything, and the readout kernel
 * for the pose kernel; results do not depend on the overlap (tests/test_gpu_api.py).
 * Errors: every call returns a ts_status; nothing throws, aborts or prints.
 */
#ifndef TS_H_
#define TS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ts_ctx ts_ctx;       /* opaque; owned by the library */
typedef struct ts_layout ts_layout; /* opaque host object: the taxel-layout builder (S0) */

typedef enum ts_status {
  TS_OK = 0,
  TS_ERR_INVALID_ARG = 1, /* NULL pointer, size out of range, inconsistent layout, ... */
  TS_ERR_CUDA = 2,        /* a CUDA runtime call or a kernel launch failed; see ts_last_error */
  TS_ERR_OOM = 3,         /* host or device allocation failed */
  TS_ERR_STATE = 4,       /* call order violated (e.g. ts_step before ts_set_geometry) */
  TS_ERR_UNSUPPORTED = 5  /* device is not sm_100 or a requested mode is not built */
} ts_status;

/* ---------------------------------------------------------------------------------------
 * S0 -- taxel-layout builder (host).  P:178 (probe = link-frame position, unit normal,
 * radius), P:182 (R_j = 0 filler slots keep batched tensors regular), P:72 / P:234 (regular
 * planar grids), P:510 (placement subsets = link filters).
 *
 * A patch is a regular nu x nv cell-centred grid of taxels on one link:
 *   x(iu,iv) = origin + ((iu+.5)/nu - .5) size_u u_axis + ((iv+.5)/nv - .5) size_v v_axis,
 *   n = u_axis x v_axis,  slot index = patch_start + iv*nu + iu  (u fastest),
 * plus an optional marker_nu x marker_nv grid of elastomer markers placed the same way
 * (marker_nu = 0: none; markers = taxels reproduces the paper's (N,3) output, Q16).
 * Limits: nu*nv <= 64 and marker_nu*marker_nv <= 64 per patch (whole patches are packed into
 * 256-slot thread blocks).  u_axis, v_axis must be unit and orthogonal to 1e-5 (the marker sum
 * is evaluated separably along u and v).
 * ------------------------------------------------------------------------------------- */
typedef struct ts_patch_desc {
  int32_t link;       /* sensor link index, 0 <= link < n_links */
  float origin[3];    /* patch centre, link frame [m] */
  float u_axis[3];
  float v_axis[3];
  float size_u, size_v; /* patch extent [m] */
  int32_t nu, nv;
  float radius;       /* probe radius R_j > 0 [m] */
  int32_t marker_nu, marker_nv;
} ts_patch_desc;

/* Read-only view of a finalised layout (host pointers owned by the layout). */
typedef struct ts_layout_view {
  int32_t n_taxels, n_patches, n_markers;
  const float* pos;       /* [T,3] link-frame positions */
  const float* nrm;       /* [T,3] link-frame unit normals */
  const float* radius;    /* [T]   0 = inactive filler */
  const int32_t* link;    /* [T] */
  const int32_t* patch;   /* [T]   -1 for trailing fillers */
  const int32_t* nbr;     /* [T,4] in-patch neighbours (-u,+u,-v,+v), -1 = none */
  const int32_t* patch_start; /* [P] */
  const int32_t* patch_nu;    /* [P] */
  const int32_t* patch_nv;    /* [P] */
  const int32_t* patch_link;  /* [P] */
  const int32_t* marker_start; /* [P] */
  const int32_t* marker_count; /* [P] */
  const float* marker_pos; /* [M,3] */
  const float* marker_nrm; /* [M,3] */
  const int32_t* marker_patch; /* [M] */
} ts_layout_view;

ts_status ts_layout_create(ts_layout** out);
/* Appends a patch; its taxels take the next nu*nv slots.  TS_ERR_INVALID_ARG on bad sizes/axes. */
ts_status ts_layout_add_patch(ts_layout* lay, const ts_patch_desc* desc);
/* Link filter: taxels (and markers' sources) on links whose mask byte is 0 become fillers
 * (radius 0).  link_mask has n_links entries.  May be called before or after finalize. */
ts_status ts_layout_filter_links(ts_layout* lay, const uint8_t* link_mask, int32_t n_links);
/* Pads with trailing filler slots up to n_taxels (>= slots used) and builds the adjacency. */
ts_status ts_layout_finalize(ts_layout* lay, int32_t n_taxels);
ts_status ts_layout_get(const ts_layout* lay, ts_layout_view* out);
ts_status ts_layout_destroy(ts_layout* lay); /* NULL is a no-op */

/* ---------------------------------------------------------------------------------------
 * Configuration (host POD, copied by ts_create).
 * ------------------------------------------------------------------------------------- */
enum { TS_HYST_OFF = 0, TS_HYST_MAXWELL = 1 /* Eq. 29-30 */, TS_HYST_ASYM = 2 /* DESIGN.md D3 */ };

/* How ts_step runs the noise chain (App. A.8): inside the step kernel (one launch after the frames kernel) or as a
 * separate kernel behind it.  AUTO = fused (the faster form for every knob combination measured).
 * Both forms compute bit-identical results. */
enum { TS_FORM_AUTO = 0, TS_FORM_FUSED = 1, TS_FORM_SPLIT = 2 };

enum {                      /* output_mask bits.  ts_step contract: every output whose bit is set must be given (non-NULL)
                               and every output whose bit is clear must be NULL; anything else is TS_ERR_INVALID_ARG */
  TS_OUT_CONTACT = 1 << 0,  /* Eq. 3   uint8 [E,T] */
  TS_OUT_DEPTH = 1 << 1,    /* Eq. 2   f32   [E,T] */
  TS_OUT_FT = 1 << 2,       /* Eq. 8-9 f32   [E,T,6] (f_x,f_y,f_z,tau_x,tau_y,tau_z), link frame */
  TS_OUT_MARKER = 1 << 3,   /* Eq. 21  f32   [E,M,3] link frame */
  TS_OUT_PROX = 1 << 4,     /* march   f32   [E,T]  P_j = r_prox - t */
  TS_OUT_FT_NOISY = 1 << 5, /* A.8     f32   [E,T,6]; needs noise_enable */
  TS_OUT_DEAD = 1 << 6,     /* Eq. 28  uint8 [E,T];   needs noise_enable */
  /* noisy readouts of the scalar sensors (Table 3: every knob of App. A.8 except crosstalk; R10);
     need noise_enable */
  TS_OUT_DEPTH_NOISY = 1 << 7,  /* f32 [E,T]   ContactDepth readout; senses with the Eq. 26 radius when radius_noise > 0 */
  TS_OUT_PROX_NOISY = 1 << 8,   /* f32 [E,T]   Proximity readout */
  TS_OUT_MARKER_NOISY = 1 << 9, /* f32 [E,M,3] Elastomer marker readout (every marker is a probe of its own) */
  TS_OUT_PROXPC = 1 << 10,      /* f32 [E,T,6] point-cloud ProximityTaxel (App. A.6, Eq. 12-17), link frame; needs
                                   ts_set_pointclouds */
  /* raycast contact-depth backend (App. A.1) on triangle meshes; needs ts_set_meshes */
  TS_OUT_DEPTH_RC = 1 << 11,    /* f32 [E,T]   deepest of sphere-triangle (R_j - dist) and ray-triangle (R_j - hit) */
  TS_OUT_NRM_RC = 1 << 12       /* f32 [E,T,3] face normal of the deepest-penetrating triangle, link frame (0 = none) */
};

typedef struct ts_config {
  int32_t n_envs;        /* E >= 1 */
  int32_t n_links;       /* L >= 1 */
  int32_t objs_per_env;  /* K >= 1 */
  int64_t env_id_base;   /* global id of env 0 (Philox counters use env_id_base + e; multi-GPU sharding);
                            0 <= env_id_base and env_id_base + n_envs <= 2^32 (the counter word is 32 bits) */
  const ts_layout* layout; /* finalised; copied to the device, may be destroyed afterwards */
  /* KinematicTaxel, Eq. 10: k_n=500 c_n=1 alpha=1.2 k_t=2 k_omega=2; mu = Coulomb cap
   * (INFINITY reproduces Eq. 8 exactly); use_velocity = 0 drops the velocity terms. */
  float k_n, c_n, alpha, k_t, k_omega, mu;
  int32_t use_velocity;
  float eta_on, eta_off; /* Eq. 3 thresholds, eta_off <= eta_on (5e-4 / 2e-4) */
  /* ElastomerTaxel dilation: s_d=100 lambda_d=8000 alpha_e=1.2 c_e=1 */
  float s_d, lambda_d, alpha_e, c_e;
  float r_prox;          /* march range [m] */
  int32_t march_steps;   /* 0..64 SDF evaluations per taxel */
  float dt;              /* physics step [s] (0.005) */
  /* noise model (App. A.8) */
  int32_t noise_enable;
  uint64_t seed;         /* Philox4x32-10 key */
  float sigma_rw_force, sigma_rw_torque; /* Eq. 25 random-walk sigma per step, channels 0-2 / 3-5 */
  int32_t hyst_mode;     /* TS_HYST_* */
  float beta, tau;       /* Maxwell (Table 12: 0.5, 0.05 s) */
  float alpha_load, alpha_unload; /* asymmetric first-order */
  float p_dead;          /* Eq. 28 Bernoulli probability, 0 <= p < 1 */
  float chi;             /* Eq. 31 crosstalk strength (4-neighbour kernel, D4) */
  uint32_t output_mask;  /* TS_OUT_* the ctx will be asked for (upper bound per step) */
  /* Remaining knobs of App. A.8 on ft -> ft_noisy (R1-R4); all zero / (1, 1) = off.  Order:
   * gain (Eq. 27) -> hysteresis -> crosstalk -> + bias + white noise + drift (Eq. 25) -> quantize (Eq. 25)
   * -> dead taxels read their stuck value (Eq. 28).  *_force act on channels 0-2, *_torque on 3-5. */
  float sigma_white_force, sigma_white_torque; /* Eq. 25 n_t ~ N(0, sigma^2), fresh every step */
  float bias_force, bias_torque;               /* Eq. 25 constant bias b */
  float quant_force, quant_torque;             /* Eq. 25 quantisation step q >= 0 (0 = off): q rint(y / q), fp32, half to even */
  float gain_min, gain_max;                    /* Eq. 27 gamma_bj ~ U[min, max] per (env, taxel, episode); 0 < min <= max */
  float stuck_min_force, stuck_max_force;      /* Eq. 28 z_bj ~ U[l, u] per (env, taxel, channel, episode), l <= u */
  float stuck_min_torque, stuck_max_torque;
  /* Eq. 11 / 31 crosstalk kernel: 0 = the 4-neighbour stencil (D4); > 0 = Gaussian G_sigma with sigma in
   * taxel pitches: separable, g[d] = exp(-d^2 / (2 sigma^2)) for |d| <= ceil(3 sigma), L1-normalised, plain
   * convolution with zeros outside the patch (R7).  sigma <= 4/3 (radius <= 4). */
  float xtalk_sigma;
  /* Eq. 26 radius noise rho >= 0 [m] (0 = off): the noisy readout senses with R~_j = max(0, R_j + eps_j),
   * eps_j ~ U[-rho, rho] per (env, taxel, episode); ft_noisy then starts from Eq. 4-9 at d~ = [R~_j - phi]_+.
   * contact, depth, ft, marker and prox keep R_j (R8). */
  float radius_noise;
  /* Eq. 25 read delay Delta_read in STEPS (0 = off) and its uniform jitter +-J steps: the readout of step n shows the
   * post-crosstalk signal of step n - max(0, Delta + k_n), k_n uniform on {-J..J}, one draw per (env, step); steps
   * before the episode began read 0; bias, white noise and drift are those of step n (R9).
   * 0 <= read_delay, read_jitter and read_delay + read_jitter <= 64; the ctx holds that many past fields
   * (24 B x n_envs x n_taxels each).  The noisy scalar readouts (TS_OUT_DEPTH_NOISY / PROX_NOISY / MARKER_NOISY) are
   * delayed by the same number of steps (their post-hysteresis signal; 8 B per taxel and 12 B per marker per slot). */
  int32_t read_delay, read_jitter;
  int32_t kernel_form;   /* TS_FORM_* (0 = AUTO) */
  /* Noisy scalar readouts (TS_OUT_DEPTH_NOISY / PROX_NOISY / MARKER_NOISY), index 0 = depth, 1 = prox, 2 = marker:
   * x = gamma * clean -> hysteresis (hyst_mode, beta, tau, alpha_*) -> y = h + bias + white + drift (Eq. 25) ->
   * quantize -> a dead probe reads its stuck value U[min, max] (Eq. 28).  gain_*, p_dead and the hysteresis are the
   * ones above; depth / prox share their taxel's gain and dead draw, a marker draws its own.  Table 12 P:523-535:
   * depth sigma 2e-4 m; proximity sigma 1e-2, rw 1e-3, quant 1e-2; elastomer sigma 1e-4 m, rw 1e-5 m, quant 1e-4 m. */
  float sn_sigma_white[3], sn_sigma_rw[3], sn_bias[3], sn_quant[3], sn_stuck_min[3], sn_stuck_max[3];
  /* Point-cloud ProximityTaxel (App. A.6): sensing radius R_j [m], k, k_s, density scalar (0.01, 300,
   * 10, 100; ts_config_default sets these).  rho_b = density / max(N_b, 1), N_b = tracked points of env b (Q27). */
  float pc_radius, pc_k, pc_ks, pc_density;
  /* Elastomer shear history (App. A.7, Eq. 22-23; R11): with shear_enable the marker output is
   * sum_i u^d_ij + sum_p u^s_pj; the tracked points p are those of ts_set_pointclouds.  A point anchors (e_p = its
   * link-frame position) when the pad's SDF at it drops below -eta_enter and un-anchors above +eta_exit;
   * u^s_pj = s_s Pi_n(z_p - e_p) h_p exp(-lambda_s |Pi_n(x_j - z_p)|^2).  P:304: s_s = 100, lambda_s = 2000,
   * eta_enter = 1e-5 m, eta_exit = 1e-4 m (ts_config_default sets these; shear_enable = 0). */
  int32_t shear_enable;
  float s_s, lambda_s, eta_enter, eta_exit;
} ts_config;

/* Fills *cfg with the paper's constants and everything else zero / off. */
void ts_config_default(ts_config* cfg);

/* ---------------------------------------------------------------------------------------
 * Geometry (per-geometry SDFs).  Arrays are HOST pointers, read before the call
 * returns (the uploads are enqueued on `stream` from a staging copy the ctx owns).
 * ------------------------------------------------------------------------------------- */
enum { TS_GEOM_NONE = 0, TS_GEOM_SPHERE = 1, TS_GEOM_BOX = 2, TS_GEOM_CAPSULE = 3, TS_GEOM_SDF = 4 };

typedef struct ts_geometry {
  const int32_t* type;  /* [E,K] TS_GEOM_* */
  const float* params;  /* [E,K,4] sphere: r | box: half-extents hx,hy,hz | capsule: r, half-length
                           (axis = local z) | SDF: grid id in params[0] */
  int32_t n_grids;      /* G >= 0 */
  int32_t grid_n;       /* N: nodes per axis, 2 <= N <= 512 (all grids alike) */
  float voxel;          /* h_v [m]; node i sits at (i - (N-1)/2) h_v on each axis: every grid is centred on its object's
                           frame origin (there is no per-grid origin[3]: an offset grid is expressed by the object pose
                           the caller passes each step, which the path applies anyway, Q26) */
  const float* grids;   /* [G,N,N,N] fp32 signed distance, x fastest: index (k*N + j)*N + i */
} ts_geometry;

/* Per-step inputs: DEVICE pointers, caller-owned, read-only.  Velocities are those of the
 * frame origin, in world axes (Eq. 4-5 with r_C, r_L = frame origins, Q4). */
typedef struct ts_step_in {
  const float* link_pos;    /* [E,L,3] */
  const float* link_quat;   /* [E,L,4] */
  const float* link_linvel; /* [E,L,3] */
  const float* link_angvel; /* [E,L,3] */
  const float* obj_pos;     /* [E,K,3] */
  const float* obj_quat;    /* [E,K,4] */
  const float* obj_linvel;  /* [E,K,3] */
  const float* obj_angvel;  /* [E,K,3] */
} ts_step_in;

/* Per-step outputs: DEVICE pointers, caller-owned, fully overwritten.  NULL = not produced.
 * Requirements: 16-byte aligned base pointers (torch / cudaMalloc allocations are). */
typedef struct ts_step_out {
  uint8_t* contact; /* [E,T]   */
  float* depth;     /* [E,T]   */
  float* ft;        /* [E,T,6] */
  float* marker;    /* [E,M,3] */
  float* prox;      /* [E,T]   */
  float* ft_noisy;  /* [E,T,6] */
  uint8_t* dead;    /* [E,T]   */
  float* depth_noisy;  /* [E,T]   */
  float* prox_noisy;   /* [E,T]   */
  float* marker_noisy; /* [E,M,3] */
  float* proxpc;       /* [E,T,6] */
  float* depth_rc;     /* [E,T]   */
  float* nrm_rc;       /* [E,T,3] */
} ts_step_out;

/* Creates a context on `cuda_device` (must be sm_100).  Allocates every device buffer the
 * path needs (layout copy, state: Schmitt bit + dead flag 1 B, hysteresis 24/48 B, drift 24 B
 * per taxel slot); nothing is allocated later except the geometry bank in ts_set_geometry. */
ts_status ts_create(const ts_config* cfg, int cuda_device, ts_ctx** out);

/* Uploads object descriptors and the SDF bank (re-tiled into the internal gather layout by a
 * kernel on `stream`).  May be called again to replace the geometry.  Synchronises `stream`
 * once before returning, so host arrays may be freed immediately. */
ts_status ts_set_geometry(ts_ctx* ctx, const ts_geometry* geo, void* stream);

/* App. A.6: "tracked links are sampled into a surface point cloud at scene reset and organized in a static BVH".
 * Here: a bank of n_clouds clouds of n_points points each, in the OBJECT frame (host fp32 [G,N,3]), and the cloud of every
 * (env, object) (host int32 [E,K], -1 = not tracked).  The ctx sorts each cloud into a uniform grid of cell size
 * pc_radius / 2 (the static spatial index; a taxel's sensing sphere meets at most 125 cells) and keeps it on the device.
 * Needed before a ts_step that asks for TS_OUT_PROXPC.  Synchronises `stream` once; may be called again. */
typedef struct ts_pointclouds {
  int32_t n_clouds, n_points;
  const float* points;
  const int32_t* cloud_id;
} ts_pointclouds;
ts_status ts_set_pointclouds(ts_ctx* ctx, const ts_pointclouds* pc, void* stream);

/* App. A.1 raycast backend: a bank of triangle meshes in the OBJECT frame -- host arrays: vert_off / tri_off
 * [n_meshes + 1] offsets into verts [sum V, 3] fp32 and tris [sum F, 3] int32 (vertex indices local to their mesh,
 * outward winding) -- and the mesh of every (env, object) (host int32 [E,K], -1 = none).  The ctx builds one bounding
 * volume hierarchy per mesh (median split, leaves of <= 4 triangles; static, because every query is made in the object
 * frame) and keeps it on the device.  Needed before a ts_step that asks for TS_OUT_DEPTH_RC / TS_OUT_NRM_RC.
 * Synchronises `stream` once; may be called again. */
typedef struct ts_meshes {
  int32_t n_meshes;
  const int32_t* vert_off;
  const int32_t* tri_off;
  const float* verts;
  const int32_t* tris;
  const int32_t* mesh_id;
} ts_meshes;
ts_status ts_set_meshes(ts_ctx* ctx, const ts_meshes* meshes, void* stream);

/* One pass of the whole hot path over all envs.  Asynchronous; never allocates. */
ts_status ts_step(ts_ctx* ctx, const ts_step_in* in, const ts_step_out* out, void* stream);

/* The same step on HOST buffers (pinned memory recommended): copies the eight inputs to
 * ctx-owned device staging, runs ts_step, and copies every non-NULL output back, all enqueued
 * on `stream` in that order.  Host buffers must stay valid until the stream reaches the end
 * of the call.  The staging (inputs + requested outputs) is allocated on the first call. */
ts_status ts_step_host(ts_ctx* ctx, const ts_step_in* host_in, const ts_step_out* host_out, void* stream);

/* Zeroes drift / hysteresis / contact state and the step count of the masked envs
 * (env_mask: DEVICE uint8 [E], NULL = all) and advances their episode, which re-draws the
 * dead-taxel mask.  Asynchronous. */
ts_status ts_reset(ts_ctx* ctx, const uint8_t* env_mask_dev, void* stream);

ts_status ts_destroy(ts_ctx* ctx); /* NULL is a no-op returning TS_OK */

/* Checkpoint / resume.  Everything a ctx carries from step to step -- the Schmitt contact bits and
 * dead flags, hysteresis and drift state, the read-delay ring, the state of the noisy scalar readouts, the shear
 * anchors, the per-env reset step / episode counters and the global step counter -- as ONE flat blob in HOST memory
 * (a fixed header followed by the arrays, each padded to 16 bytes).  Layout, geometry, point clouds and meshes are NOT part of it: the blob
 * restores into a ctx created with the same layout and configuration (sizes and section set are checked; anything else
 * returns TS_ERR_INVALID_ARG and leaves the ctx untouched), after which stepping continues bit for bit as in the ctx it
 * was taken from.  Both calls enqueue their copies on `stream` and synchronise it once before returning.
 * ts_state_bytes: size of the blob for this ctx (it depends on the configuration only).
 * ts_get_state:   host_buf [capacity >= ts_state_bytes] is filled.
 * ts_set_state:   host_buf [bytes] as written by ts_get_state. */
ts_status ts_state_bytes(const ts_ctx* ctx, uint64_t* bytes);
ts_status ts_get_state(ts_ctx* ctx, void* host_buf, uint64_t capacity, void* stream);
ts_status ts_set_state(ts_ctx* ctx, const void* host_buf, uint64_t bytes, void* stream);

/* Allocation-free entry point, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it).  It needs no ctx and calls no cudaMalloc, cudaFree or allocating library routine:
 * the contact depth d = [R_j - phi(x_o)]_+ (App. A.1-A.2, Eq. 1-2) of every (env, taxel) against ONE analytic primitive
 * per env (TS_GEOM_SPHERE / BOX / CAPSULE; any other type reads as "no object", depth 0), the same arithmetic as the
 * depth output of the ctx path.  Its only scratch, the relative pose of every (env, link), lives in a static device array
 * of TS_STATIC_SCRATCH_BYTES (8 MiB) inside the library, which every GPU that loads the library holds until the process
 * exits: n_envs * n_links <= TS_STATIC_MAX_FRAMES, anything larger returns TS_ERR_INVALID_ARG with the limit in
 * the error text (read it with a NULL ctx below).  Runs on the CURRENT device, on `stream`; two kernels are enqueued, nothing
 * synchronises.  All calls on a device share that array: calls on one stream are ordered and each call overwrites what it
 * reads (nothing has to be cleared between calls), but calls that overlap on the GPU (different streams without an
 * event between them) race on it.
 * All pointers are DEVICE pointers, caller-owned, row-major fp32 / int32:
 *   taxel_pos [T,3] link-frame positions, taxel_radius [T] R_j (<= 0: filler, depth 0), taxel_link [T] link of each
 *   taxel (outside [0, n_links): depth 0)  -- the pos / radius / link arrays of ts_layout_view, copied to the device;
 *   link_pos [E,L,3], link_quat [E,L,4] (w,x,y,z), obj_pos [E,3], obj_quat [E,4];
 *   geom_type [E] int32, geom_params [E,4] (16-byte aligned) as in ts_geometry with objs_per_env = 1;
 *   depth [E,T] out. */
enum { TS_STATIC_SCRATCH_BYTES = 8 << 20, TS_STATIC_MAX_FRAMES = (8 << 20) / 96 };
ts_status ts_depth_static(int32_t n_envs, int32_t n_links, int32_t n_taxels, const float* taxel_pos, const float* taxel_radius,
                          const int32_t* taxel_link, const float* link_pos, const float* link_quat, const float* obj_pos,
                          const float* obj_quat, const int32_t* geom_type, const float* geom_params, float* depth, void* stream);

/* Last error text of this ctx (with a NULL ctx: of the last failed ctx-free call of this thread, i.e. ts_create or
 * ts_depth_static).  Never NULL. */
const char* ts_last_error(const ts_ctx* ctx);

/* Introspection used by the binding and the bench. */
int32_t ts_n_taxels(const ts_ctx* ctx);
int32_t ts_n_markers(const ts_ctx* ctx);
/* Number of kernel launches one ts_step enqueues with the ctx's current configuration. */
int32_t ts_launches_per_step(const ts_ctx* ctx);
/* Kernel timing.  With recording on, ts_step brackets its launches with CUDA events on the step's own stream (a fixed
 * pool of TS_TIMING_MAX_STEPS slots created when recording is switched on; further steps are not recorded, nothing is
 * ever allocated inside ts_step).  ts_kernel_time_ms synchronises the recorded events, returns the MEAN duration in ms
 * of all kernels of a step over the steps recorded since the last call, and sets recording to `enable`: 0 = off,
 * 1 = one pair of events around the kernels of a step (the whole step lands in the step-kernel column below),
 * 2 = events between the kernels as well (per-kernel durations; the extra records cost a few microseconds per step).
 * ts_kernel_times_ms (call it BEFORE ts_kernel_time_ms, which clears the record) copies the per-step durations:
 * out_ms[4 * i + 0] = frames kernel, + 1 = step kernel, + 2 = separate noise kernel (0 when fused), from the CUDA
 * events, and + 3 = the step's span on the DEVICE-SIDE clock: %globaltimer at the start of the first block of the
 * frames kernel to %globaltimer at the end of the last block of the step's last kernel (written by the kernels
 * themselves while recording is on), for i < min(recorded, capacity); *n_steps gets the number recorded. */
enum { TS_TIMING_MAX_STEPS = 4096 };
ts_status ts_kernel_time_ms(ts_ctx* ctx, int32_t enable, float* mean_ms, int32_t* n_steps);
ts_status ts_kernel_times_ms(ts_ctx* ctx, float* out_ms, int32_t capacity, int32_t* n_steps);
/* Mean duration in ms of the frames kernel + the step kernel over the steps the last ts_kernel_time_ms call averaged;
 * the remainder of its mean_ms is the separate noise kernel (0 when the noise chain is fused). */
float ts_first_kernel_time_ms(const ts_ctx* ctx);

const char* ts_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TS_H_ */
