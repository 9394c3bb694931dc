// Internal declarations shared by the host side (ts_layout.cpp, ts_api.cu) and the kernels
// (ts_kernels.cu).  Not part of the public ABI.
#ifndef TS_INTERNAL_H_
#define TS_INTERNAL_H_

#include <cstdint>
#include <vector>

#include <vector_types.h>  // float4 (host and device)

#include "../../include/ts.h"

#define TS_MAX_PATCH_TAXELS 64  // one warp owns a patch: 2 taxel slots per lane

struct ts_layout {
  bool finalized = false;
  int n_taxels = 0;
  std::vector<float> pos, nrm, radius, radius_cfg;
  std::vector<int32_t> link, patch, nbr;
  std::vector<int32_t> patch_start, patch_nu, patch_nv, patch_link, marker_start, marker_count;
  std::vector<float> patch_eps;  // pitch along u (epsilon of Eq. 20, Q15)
  std::vector<float> marker_pos, marker_nrm;
  std::vector<int32_t> marker_patch;
};

// Device-side patch record (two 16-byte loads per warp).
struct TsPatch {
  int32_t start;   // first taxel slot
  int32_t n;       // taxel slots in the patch (<= 64)
  int32_t nu;      // grid width (u fastest); fillers: nu = n
  int32_t link;    // sensor link, -1 = filler patch (all slots inactive)
  int32_t mstart;  // first marker
  int32_t mcount;  // markers (<= 64)
  float eps;       // Eq. 20 epsilon
  int32_t pad;
};

// Kernel parameters of one step (passed by value).
struct TsStepParams {
  int32_t E, L, K, T, P, M;
  uint32_t env_id_base;
  // layout
  const float4* tx_pos;  // [T] (x, y, z, R_j)
  const float4* tx_nrm;  // [T] (nx, ny, nz, 0)
  const TsPatch* patches;  // [P]
  const float4* mk_pos;  // [M]
  const float4* mk_nrm;  // [M]
  // geometry
  const int32_t* g_type;   // [E,K]
  const float4* g_params;  // [E,K]
  const float4* bank;      // re-tiled SDF bank (see ts_kernels.cu, "bank layout")
  int32_t grid_n;
  float voxel, inv_voxel, grid_origin;
  double inv_voxel_d;  // 1 / (double)voxel, for the fp64 first query
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
  // state
  uint8_t* st_flags;          // [E,T] bit0 Schmitt, bit1 dead
  float4* st_hyst;            // [E,P,nh,32] float4, nh = 3 (asym) / 6 (maxwell)
  float4* st_drift;           // [E,P,3,32] float4
  const uint32_t* reset_step; // [E]
  const uint32_t* episode;    // [E]
  uint32_t gstep;
  // physics
  float k_n, c_n, alpha, k_t, k_omega, mu, eta_on, eta_off;
  int32_t use_velocity;
  float s_d, lambda_d, alpha_e, c_e, inv_gbar;
  float r_prox;
  int32_t march_steps;
  // noise
  int32_t noise_enable, hyst_mode;
  uint32_t seed_lo, seed_hi;
  float sigma_f, sigma_t, beta, decay, alpha_load, alpha_unload, chi;
};

// launchers (ts_kernels.cu)
int ts_launch_step(const TsStepParams& p, void* stream);
int ts_launch_retile(const float* src_linear, float4* dst, int n_grids, int N, void* stream);
int ts_launch_reset_counters(uint32_t* reset_step, uint32_t* episode, const uint8_t* mask, int E, uint32_t gstep,
                             void* stream);
int ts_launch_reset_state(const TsStepParams& p, const uint8_t* mask, uint32_t dead_threshold, int nh, void* stream);
unsigned long long ts_bank_elems_per_grid(int N);

#endif  // TS_INTERNAL_H_
