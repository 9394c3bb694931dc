// Internal declarations shared by the host side (ts_layout.cpp, ts_api.cu) and the kernels
// (ts_kernels.cu).  Not part of the public ABI.
#ifndef TS_INTERNAL_H_
#define TS_INTERNAL_H_

#include <cstdint>
#include <vector>

#include <vector_types.h>  // float4 (host and device)

#include "../../include/ts.h"

#define TS_MAX_PATCH_TAXELS 64   // taxels (and markers) per patch
#ifndef TS_BLOCK
#define TS_BLOCK 256             // threads per block = taxel slots per patch group
#endif
#define TS_MAX_GROUP_PATCHES 32  // patches per group
#define TS_INL_GROUPS 16         // group records / link ids carried inside the kernel parameters
#define TS_INL_LINKS 192
#ifndef TS_CHUNK
#define TS_CHUNK (3 * TS_BLOCK / 2)  // marker pass-1 items / markers per chunk
#endif

struct ts_layout {
  bool finalized = false;
  int n_taxels = 0;
  std::vector<ts_patch_desc> desc;  // as given to ts_layout_add_patch
  std::vector<float> pos, nrm, radius, radius_cfg;
  std::vector<int32_t> link, patch, nbr;
  std::vector<int32_t> patch_start, patch_nu, patch_nv, patch_link, marker_start, marker_count;
  std::vector<float> patch_eps;  // pitch along u (epsilon of Eq. 20, Q15)
  std::vector<float> marker_pos, marker_nrm;
  std::vector<int32_t> marker_patch;
};

// Device-side patch record (112 bytes).
struct TsPatch {
  int32_t start;   // first taxel slot
  int32_t n;       // taxel slots in the patch
  int32_t nu, nv;  // taxel grid (u fastest); fillers: nu = n, nv = 1
  int32_t link;    // sensor link, -1 = filler patch (all slots inactive)
  int32_t mstart;  // first marker
  int32_t mnu, mnv;  // marker grid (0 = none)
  float eps;       // Eq. 20 epsilon
  int32_t tab;     // offset (doubles) of this patch's separable tables in mk_tab
  int32_t i1off;   // first pass-1 item of this patch (index into mk_item1)
  int32_t direct;  // 1 = direct (non-separable) marker sum
  float4 ua, va, na;  // u axis (w = pad extent size_u), v axis (w = size_v), normal (link frame)
  float4 ctr;         // pad centre (link frame); the pad is the elastomer surface of Eq. 22's SDF
};

// A group = consecutive patches whose taxel slots fit one block.
struct TsGroup {
  int32_t start, count;    // taxel slots [start, start + count)
  int32_t patch0, npatch;  // patches [patch0, patch0 + npatch)
  int32_t chunk0, nchunk;  // marker chunks [chunk0, chunk0 + nchunk)
  int32_t mstart, mcount;  // markers of the group (contiguous)
};

// A marker chunk = consecutive patches of one group whose pass-1 items and markers fit one block.
struct TsChunk {
  int32_t i1_begin, i1_end;  // pass-1 items (a, q) in mk_item1
  int32_t m_begin, m_end;    // markers (pass-2 items) in mk_item2
  int32_t lp_begin, lp_end;  // group-local patch range
  int32_t pad0, pad1;
};

// Uniform grid over one tracked point cloud (object frame), cell size = the sensing radius.
// Uniform grid of a tracked point cloud: cell = sensing radius / TS_PC_REACH, so the points within the radius of a
// query lie in the (2 * TS_PC_REACH + 1)^3 cells around its own.  Finer cells scan fewer points outside the sphere
// (candidates per in-sphere point: 6.4 with reach 1, 3.7 with reach 2) at the price of more, shorter runs.
#ifndef TS_PC_REACH
#define TS_PC_REACH 2
#endif
struct TsPcGrid {
  float ox, oy, oz, inv_cell;  // cell (i, j, k) covers origin + (i..i+1, j..j+1, k..k+1) * cell
  int32_t nx, ny, nz;
  int32_t cell0;               // offset of this cloud's cell_start array in pc_cell
  int32_t pt0;                 // offset of this cloud's points in pc_pts
  int32_t pad[3];
};

// Kernel parameters of one step (passed by value).
struct TsStepParams {
  int32_t E, L, K, T, P, M, G, Tp;
  int32_t frames_per_group;  // max patches per group (shared-memory frames = this * K)
  uint32_t env_id_base;
  // layout
  const float4* tx_pos;   // [T] (x, y, z, R_j); R_j = 0 for every inactive slot
  const int32_t* tx_patch; // [T] global patch index of each slot (fillers: their filler patch)
  const int32_t* tx_meta; // [T] bits 0-7 group-local patch index, 8-15 patch nu, 16-19 has -u/+u/-v/+v neighbour
  const TsPatch* patches; // [P]
  const TsGroup* groups;  // [G]
  const TsChunk* chunks;
  const int32_t* grp_link;  // [G][TS_MAX_GROUP_PATCHES] sensor link of each patch of a group (-1 = filler)
  const int32_t* mk_item1;  // packed lp | a << 8 | q << 16
  const int32_t* mk_item2;  // [M] packed lp | a << 8 | b << 16
  const double* mk_tab;     // per patch: GU[mnu][nu], DU[mnu][nu], GV[mnv][nv], DV[mnv][nv]
  const double* mk_tab8;    // per patch [4][8][8], zero-padded: GU[a][p], DU[a][p], GV[b][q], DV[b][q] (DMMA marker path)
  int32_t mk_mma;           // 1 = every patch with markers has nu, nv, mnu, mnv <= 8 and a separable sum: DMMA path
  int32_t s_bytes;          // bytes of the shared-memory region S / bufB (9 KB with the generic marker path, 6 KB with DMMA)
  const float4* mk_pos;   // [M]
  const float4* mk_nrm;   // [M]
  // geometry
  const int32_t* g_type;   // [E,K]
  const float4* g_params;  // [E,K]
  unsigned long long* clock;  // NULL, or this step's {first block start, last block end} %globaltimer stamps [ns]
  void* frames_g;          // [E][P*K] FrameS (ts_kernels.cu): relative poses of every (env, patch, object), written by
                           // ts_frames_kernel at the start of the step, bulk-copied (TMA) into shared memory by each block
  const int32_t* patch_link;  // [P] sensor link of each patch (-1 = filler)
  const int32_t* env_perm; // [E] block -> env: envs ordered by (geometry type, grid id) so that the blocks resident at any
                           // time gather from ONE grid of the bank (L2-resident) and run one march loop; NULL = identity
  const float4* bank;      // re-tiled SDF bank (see ts_kernels.cu, "bank layout")
  int32_t grid_n;
  float voxel, inv_voxel;
  double inv_voxel_d;      // 1 / (double)voxel
  unsigned long long grid_stride;  // float4 elements per grid
  // inputs
  const float *link_pos, *link_quat, *link_linvel, *link_angvel;
  const float *obj_pos, *obj_quat, *obj_linvel, *obj_angvel;
  // outputs (NULL = skip)
  uint8_t* contact;
  float* depth;
  float* ft;
  float* marker;
  float* prox;
  float* ft_noisy;
  uint8_t* dead;
  // noisy scalar readouts (R10): outputs, the perturbed depth the step kernel leaves for them (Eq. 26), their state
  float* depth_noisy;
  float* prox_noisy;
  float* marker_noisy;
  float* depth_pert;          // [E,T] d~ = [R~_j - phi]_+ (written by the step kernel when radius noise is on), else NULL
  float4* sn_h;               // [E,T] hysteresis of (depth, prox): Maxwell (xi_d, xprev_d, xi_p, xprev_p), ASYM (y_d, y_p, -, -)
  float2* sn_d;               // [E,T] drift of (depth, prox)
  float* sm_h;                // [E,M,6] marker hysteresis: 3 x (xi | y), 3 x x_prev
  float* sm_d;                // [E,M,3] marker drift
  float sn_sigma_white[3], sn_sigma_rw[3], sn_bias[3], sn_quant[3], sn_stuck_min[3], sn_stuck_max[3];
  uint32_t dead_thr;          // floor(p_dead 2^32)
  // point-cloud ProximityTaxel (A.6)
  float* proxpc;              // [E,T,6] output
  const float4* pc_pts;       // clouds sorted by grid cell: (x, y, z, -) in the object frame
  const int32_t* pc_cell;     // per cloud: cell_start[ncell + 1] (indices into pc_pts), concatenated
  const struct TsPcGrid* pc_grid;  // [G]
  const int32_t* pc_id;       // [E,K] cloud of each object, -1 = none
  int32_t pc_n;               // points per cloud
  int32_t pc_np;              // pc_n rounded up to 16: stride of the shear anchor rows (16-byte aligned flag rows)
  float pc_radius, pc_k, pc_ks, pc_density;
  // raycast depth backend (A.1): BVH nodes and leaf-ordered triangles of every mesh
  float* depth_rc;            // [E,T]
  float* nrm_rc;              // [E,T,3]
  const float4* rc_nodes;     // 2 float4 per node: (lo.xyz, first triangle | left child), (hi.xyz, count > 0 | -right child)
  const float4* rc_tri;       // 3 float4 per triangle (vertices a, b, c), in leaf order
  const int32_t* rc_root;     // [G] root node of each mesh
  const int32_t* rc_id;       // [E,K] mesh of each object, -1 = none
  // elastomer shear history (Eq. 22): anchors per (env, patch, object, tracked point)
  uint8_t* sh_on;             // [E,P,K,Np] anchored?  (Np = pc_np)
  int32_t* sh_cnt;            // [E,P,K] number of anchored points (lets a pad with none skip the flag scan)
  float4* sh_e;               // [E,P,K,Np] anchor relative to the pad centre (link frame); only read where sh_on is set
  const float4* pc_raw;       // [G,N] tracked points in their original order (the grid-sorted copy serves the proximity query)
  int32_t shear_enable;
  float s_s, lambda_s, eta_enter, eta_exit;
  // read delay of the noisy scalar readouts (R10): the last rd_S post-hysteresis signals
  float2* sn_ring;            // [E, rd_S, T] (depth, prox); NULL = no delay or outputs not requested
  float* sm_ring;             // [E, rd_S, M, 3] markers
  // state
  uint8_t* st_flags;          // [E,T] bit0 Schmitt, bit1 dead
  float* st_hyst;             // [E,nh/2,Tp] float2 channel pairs, nh = 6 (asym: y) / 12 (maxwell: xi then x_prev)
  float* st_drift;            // [E,3,Tp] float2 channel pairs
  const uint32_t* reset_step; // [E]
  const uint32_t* episode;    // [E]
  uint32_t gstep;
  // physics
  float k_n, c_n, alpha, k_t, k_omega, mu, eta_on, eta_off;
  int32_t use_velocity;
  float s_d, lambda_d, alpha_e, c_e;
  double inv_gbar;            // 1 / g_bar = sqrt(2 lambda_d) e^{1/2}
  float r_prox;
  int32_t march_steps;
  // noise
  int32_t noise_enable, hyst_mode;
  uint32_t seed_lo, seed_hi;
  float sigma_f, sigma_t, beta, decay, alpha_load, alpha_unload, chi;
  // remaining A.8 knobs (Eq. 25, 27, 28); ext = 1 selects the kernel variant that evaluates them
  int32_t ext;
  float sigma_wf, sigma_wt, bias_f, bias_t, quant_f, quant_t, gain_min, gain_max;
  float stuck_lo_f, stuck_hi_f, stuck_lo_t, stuck_hi_t;
  int32_t xt_r;     // Gaussian crosstalk radius ceil(3 sigma) <= 4; 0 = 4-neighbour stencil
  float xt_w[5];    // L1-normalised 1-D weights g[|d|], d = 0..xt_r
  float rho;        // Eq. 26 radius noise (0 = off or noise off)
  float* ft_pert;   // two-kernel variant with rho != 0: [E,T,6] Eq. 4-9 at the perturbed depth, else NULL
  int32_t rd_delay, rd_jitter, rd_S;  // Eq. 25 read delay (steps), jitter, ring slots S = delay + jitter (0 = off)
  float* st_ring;   // [E,S,3,Tp] float2 channel pairs: post-crosstalk fields of the last S steps
  // Small layouts carry their group records and per-group link ids in the parameter space itself (constant
  // bank: a few cycles) so that a block's first dependent global load is already the pose row.
  int32_t inl;                             // 1 = the two tables below are valid
  int32_t inl_stride;                      // link ids per group in inl_link (= frames_per_group)
  TsGroup inl_grp[TS_INL_GROUPS];
  int32_t inl_link[TS_INL_LINKS];
};

// launchers (ts_kernels.cu)
int ts_launch_step(const TsStepParams& p, int fused_noise, void* stream);
int ts_launch_noise(const TsStepParams& p, void* stream);
int ts_launch_frames(const TsStepParams& p, void* stream);
int ts_launch_scalar_noise(const TsStepParams& p, void* stream);
int ts_launch_proxpc(const TsStepParams& p, void* stream);
int ts_launch_shear(const TsStepParams& p, void* stream);
int ts_launch_raycast(const TsStepParams& p, void* stream);
int ts_launch_reset_shear(const TsStepParams& p, const uint8_t* mask, void* stream);
int ts_launch_reset_scalar(const TsStepParams& p, const uint8_t* mask, void* stream);
unsigned long long ts_frame_bytes();
int ts_launch_retile(const float* src_linear, float4* dst, int n_grids, int N, void* stream);
int ts_launch_reset_counters(uint32_t* reset_step, uint32_t* episode, const uint8_t* mask, int E, uint32_t gstep,
                             void* stream);
int ts_launch_reset_state(const TsStepParams& p, const uint8_t* mask, uint32_t dead_threshold, int nh, void* stream);
unsigned long long ts_bank_elems_per_grid(int N);
unsigned long long ts_step_smem_bytes(const TsStepParams& p);
int ts_prepare_kernels(int device, int smem_bytes);
// ts_depth_static: pose kernel + depth kernel on the current device with the poses in the library's static scratch
// array (sizes as in include/ts.h: TS_STATIC_SCRATCH_BYTES, TS_STATIC_MAX_FRAMES); returns a cudaError_t.
int ts_static_depth_launch(int E, int L, int T, const float* taxel_pos, const float* taxel_radius, const int32_t* taxel_link,
                           const float* link_pos, const float* link_quat, const float* obj_pos, const float* obj_quat,
                           const int32_t* geom_type, const float* geom_params, float* depth, void* stream);

#endif  // TS_INTERNAL_H_
