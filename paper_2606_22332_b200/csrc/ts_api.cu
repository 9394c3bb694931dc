// C ABI of include/ts.h: context, validation, uploads, launches.  No compute happens here.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "ts_internal.h"

#ifndef TS_DEFAULT_SPLIT
#define TS_DEFAULT_SPLIT 0
#endif

struct ts_ctx {
  int device = 0;
  ts_config cfg{};
  int T = 0, P = 0, M = 0, nh = 0, G = 0, Tp = 0, frames_per_group = 1;
  bool have_geometry = false;
  uint32_t gstep = 0;
  uint32_t dead_thr = 0;
  // device buffers
  float4 *tx_pos = nullptr, *mk_pos = nullptr, *mk_nrm = nullptr;
  int32_t* tx_meta = nullptr;
  TsPatch* patches = nullptr;
  TsGroup* groups = nullptr;
  TsChunk* chunks = nullptr;
  int32_t *mk_item1 = nullptr, *mk_item2 = nullptr, *grp_link = nullptr;
  std::vector<TsGroup> h_groups;   // host copies for the inline parameter tables
  std::vector<int32_t> h_glink;
  double* mk_tab = nullptr;
  double* mk_tab8 = nullptr;   // zero-padded 8 x 8 separable tables (DMMA marker path)
  bool mk_mma = false;
  int32_t* g_type = nullptr;
  float4* g_params = nullptr;
  void* frames_g = nullptr;       // [E][P*K] relative-pose frames of the current step (ts_frames_kernel -> ts_step_kernel)
  int32_t* patch_link = nullptr;  // [P]
  int32_t* env_perm = nullptr;  // block -> env order of the step kernel (sorted by geometry; set by ts_set_geometry)
  float4* bank = nullptr;
  size_t bank_bytes = 0;
  float* bank_stage = nullptr;  // linear copy of the bank the re-tiling kernel reads (kept between ts_set_geometry calls)
  size_t bank_stage_bytes = 0;
  std::vector<int32_t> h_perm;  // host copy of env_perm (source of the asynchronous upload)
  int grid_n = 2, n_grids = 0;
  float voxel = 1.f;
  uint8_t* st_flags = nullptr;
  float *st_hyst = nullptr, *st_drift = nullptr;
  uint32_t *reset_step = nullptr, *episode = nullptr;
  // device staging of ts_step_host
  float* stage_in[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  void* stage_out[13] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  // raycast depth backend (A.1): BVH nodes, leaf-ordered triangles, root per mesh, mesh of each (env, object)
  float4* rc_nodes = nullptr; float4* rc_tri = nullptr; int32_t* rc_root = nullptr; int32_t* rc_id = nullptr; bool have_mesh = false;
  // point-cloud ProximityTaxel (A.6): clouds sorted by grid cell, cell starts, grid records, cloud of each (env, object)
  float4* pc_pts = nullptr; int32_t* pc_cell = nullptr; TsPcGrid* pc_grid = nullptr; int32_t* pc_id = nullptr;
  int32_t* tx_patch = nullptr;
  int pc_n = 0; bool have_pc = false;
  uint8_t* sh_on = nullptr; float4* sh_e = nullptr; float4* pc_raw = nullptr; int32_t* sh_cnt = nullptr;   // elastomer shear history (Eq. 22)
  // noisy scalar readouts (R10): state, the perturbed depth (Eq. 26), scratch copies of clean inputs the caller did not ask for
  float4* sn_h = nullptr; float2* sn_d = nullptr; float *sm_h = nullptr, *sm_d = nullptr;
  float *depth_pert = nullptr, *sc_depth = nullptr, *sc_prox = nullptr, *sc_marker = nullptr;
  float2* sn_ring = nullptr; float* sm_ring = nullptr;   // read-delay rings of the scalar readouts (R10)
  // timing of the main kernel
  bool timing = false;
  bool timing_detail = false;   // events between the kernels of a step too (enable = 2)
  std::vector<cudaEvent_t> ev;  // 4 per step: before the frames kernel, after it, after the step kernel, after the noise kernel;
                                // fixed pool of 4 * TS_TIMING_MAX_STEPS created when recording is switched on
  float last_first_kernel_ms = 0.f;
  bool fused = true;            // one fused launch (default) or geometry + noise kernels (TS_SPLIT=1)
  float* ft_scratch = nullptr;  // clean ft for the noise kernel when the caller does not ask for ft
  float* st_ring = nullptr;       // Eq. 25 read delay: the last read_delay + read_jitter post-crosstalk fields
  float* ft_scratch_r = nullptr;  // two-kernel variant with radius noise: Eq. 4-9 at the perturbed depth (Eq. 26)
  size_t ev_used = 0;
  unsigned long long* clock_buf = nullptr;  // [TS_TIMING_MAX_STEPS][2] device-side clock stamps (allocated with the event pool)
  std::string err;
};

namespace {
thread_local std::string g_create_err;

ts_status fail(ts_ctx* c, ts_status s, const std::string& msg) {
  if (c) c->err = msg; else g_create_err = msg;
  return s;
}
ts_status cuda_fail(ts_ctx* c, cudaError_t e, const char* what) {
  return fail(c, e == cudaErrorMemoryAllocation ? TS_ERR_OOM : TS_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define TS_CUDA(ctx, call)                                   \
  do {                                                       \
    cudaError_t e_ = (call);                                 \
    if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call); \
  } while (0)

struct DeviceGuard {
  int prev = -1;
  explicit DeviceGuard(int dev) { cudaGetDevice(&prev); if (prev != dev) cudaSetDevice(dev); else prev = -1; }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

void free_all(ts_ctx* c) {
  cudaFree(c->tx_pos); cudaFree(c->tx_meta); cudaFree(c->mk_pos); cudaFree(c->mk_nrm); cudaFree(c->patches);
  cudaFree(c->groups); cudaFree(c->chunks); cudaFree(c->mk_item1); cudaFree(c->mk_item2); cudaFree(c->mk_tab); cudaFree(c->mk_tab8); cudaFree(c->grp_link);
  cudaFree(c->g_type); cudaFree(c->g_params); cudaFree(c->env_perm); cudaFree(c->frames_g); cudaFree(c->patch_link); cudaFree(c->bank); cudaFree(c->bank_stage); cudaFree(c->st_flags); cudaFree(c->st_hyst);
  cudaFree(c->st_drift); cudaFree(c->reset_step); cudaFree(c->episode); cudaFree(c->ft_scratch); cudaFree(c->ft_scratch_r); cudaFree(c->st_ring);
  cudaFree(c->rc_nodes); cudaFree(c->rc_tri); cudaFree(c->rc_root); cudaFree(c->rc_id);
  cudaFree(c->sh_on); cudaFree(c->sh_e); cudaFree(c->pc_raw); cudaFree(c->sh_cnt);
  cudaFree(c->pc_pts); cudaFree(c->pc_cell); cudaFree(c->pc_grid); cudaFree(c->pc_id); cudaFree(c->tx_patch);
  cudaFree(c->sn_h); cudaFree(c->sn_d); cudaFree(c->sm_h); cudaFree(c->sm_d); cudaFree(c->depth_pert); cudaFree(c->sc_depth);
  cudaFree(c->sc_prox); cudaFree(c->sc_marker); cudaFree(c->sn_ring); cudaFree(c->sm_ring);
  for (float* q : c->stage_in) cudaFree(q);
  for (void* q : c->stage_out) cudaFree(q);
  for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
  cudaFree(c->clock_buf);
}

// 1 = a knob beyond the four of configs 4-5 is set: selects the kernel variants that carry them (HM | 4).
int cfg_ext(const ts_config& g) {
  return (g.noise_enable && (g.read_delay != 0 || g.read_jitter != 0 || g.radius_noise != 0.f || g.xtalk_sigma != 0.f || g.sigma_white_force != 0.f || g.sigma_white_torque != 0.f || g.bias_force != 0.f || g.bias_torque != 0.f ||
                              g.quant_force != 0.f || g.quant_torque != 0.f || g.gain_min != 1.f || g.gain_max != 1.f ||
                              g.stuck_min_force != 0.f || g.stuck_max_force != 0.f || g.stuck_min_torque != 0.f ||
                              g.stuck_max_torque != 0.f)) ? 1 : 0;
}

void fill_params(const ts_ctx* c, TsStepParams& p) {
  const ts_config& g = c->cfg;
  std::memset(&p, 0, sizeof(p));
  p.E = g.n_envs; p.L = g.n_links; p.K = g.objs_per_env; p.T = c->T; p.P = c->P; p.M = c->M;
  p.G = c->G; p.Tp = c->Tp; p.frames_per_group = c->frames_per_group;
  p.groups = c->groups; p.chunks = c->chunks; p.mk_item1 = c->mk_item1; p.mk_item2 = c->mk_item2;
  p.mk_tab = c->mk_tab; p.grp_link = c->grp_link;
  p.mk_tab8 = c->mk_tab8; p.mk_mma = c->mk_mma ? 1 : 0;
  p.s_bytes = c->mk_mma ? (int32_t)(sizeof(float) * 6 * TS_BLOCK) : (int32_t)(sizeof(double) * 3 * TS_CHUNK);
  p.inl = 0; p.inl_stride = c->frames_per_group;
  if (c->G <= TS_INL_GROUPS && c->G * c->frames_per_group <= TS_INL_LINKS && (int)c->h_groups.size() == c->G) {
    p.inl = 1;
    for (int g = 0; g < c->G; ++g) {
      p.inl_grp[g] = c->h_groups[g];
      for (int l = 0; l < c->frames_per_group; ++l) p.inl_link[g * c->frames_per_group + l] = c->h_glink[(size_t)g * TS_MAX_GROUP_PATCHES + l];
    }
  }
  p.env_id_base = (uint32_t)g.env_id_base;
  p.tx_pos = c->tx_pos; p.tx_meta = c->tx_meta; p.patches = c->patches; p.mk_pos = c->mk_pos; p.mk_nrm = c->mk_nrm;
  p.g_type = c->g_type; p.g_params = c->g_params; p.bank = c->bank; p.env_perm = c->env_perm; p.frames_g = c->frames_g; p.patch_link = c->patch_link;
  p.grid_n = c->grid_n; p.voxel = c->voxel; p.inv_voxel = 1.0f / c->voxel; p.inv_voxel_d = 1.0 / (double)c->voxel;
  p.grid_stride = ts_bank_elems_per_grid(c->grid_n);
  p.st_flags = c->st_flags; p.st_hyst = c->st_hyst; p.st_drift = c->st_drift;
  p.reset_step = c->reset_step; p.episode = c->episode; p.gstep = c->gstep;
  p.k_n = g.k_n; p.c_n = g.c_n; p.alpha = g.alpha; p.k_t = g.k_t; p.k_omega = g.k_omega; p.mu = g.mu;
  p.eta_on = g.eta_on; p.eta_off = g.eta_off; p.use_velocity = g.use_velocity;
  p.s_d = g.s_d; p.lambda_d = g.lambda_d; p.alpha_e = g.alpha_e; p.c_e = g.c_e;
  // 1 / g_bar, g_bar = e^{-1/2} / sqrt(2 lambda_d)
  p.inv_gbar = std::sqrt(2.0 * (double)g.lambda_d) / std::exp(-0.5);
  p.r_prox = g.r_prox; p.march_steps = g.march_steps;
  p.noise_enable = g.noise_enable; p.hyst_mode = g.noise_enable ? g.hyst_mode : TS_HYST_OFF;
  p.seed_lo = (uint32_t)(g.seed & 0xffffffffu); p.seed_hi = (uint32_t)(g.seed >> 32);
  p.sigma_f = g.sigma_rw_force; p.sigma_t = g.sigma_rw_torque; p.beta = g.beta;
  p.decay = (g.tau > 0.f) ? (float)std::exp(-(double)g.dt / (double)g.tau) : 0.f;   // Eq. 29
  p.alpha_load = g.alpha_load; p.alpha_unload = g.alpha_unload; p.chi = g.chi;
  p.sigma_wf = g.sigma_white_force; p.sigma_wt = g.sigma_white_torque; p.bias_f = g.bias_force; p.bias_t = g.bias_torque;
  p.quant_f = g.quant_force; p.quant_t = g.quant_torque; p.gain_min = g.gain_min; p.gain_max = g.gain_max;
  p.stuck_lo_f = g.stuck_min_force; p.stuck_hi_f = g.stuck_max_force; p.stuck_lo_t = g.stuck_min_torque; p.stuck_hi_t = g.stuck_max_torque;
  p.xt_r = 0;
  for (int d = 0; d < 5; ++d) p.xt_w[d] = 0.f;
  if (g.noise_enable && g.xtalk_sigma > 0.f) {  // Eq. 11 / 31, R7: separable L1-normalised Gaussian taps
    const double sg = (double)g.xtalk_sigma;
    const int r = (int)std::ceil(3.0 * sg);
    double norm = 0.0;
    for (int d = -r; d <= r; ++d) norm += std::exp(-(double)(d * d) / (2.0 * sg * sg));
    p.xt_r = r;
    for (int d = 0; d <= r && d < 5; ++d) p.xt_w[d] = (float)(std::exp(-(double)(d * d) / (2.0 * sg * sg)) / norm);
  }
  p.rd_delay = g.noise_enable ? g.read_delay : 0; p.rd_jitter = g.noise_enable ? g.read_jitter : 0;
  p.rd_S = p.rd_delay + p.rd_jitter; p.st_ring = c->st_ring;
  p.rho = g.noise_enable ? g.radius_noise : 0.f;
  p.ft_pert = (p.rho != 0.f && !c->fused) ? c->ft_scratch_r : nullptr;
  p.ext = cfg_ext(g);
  p.sn_h = c->sn_h; p.sn_d = c->sn_d; p.sm_h = c->sm_h; p.sm_d = c->sm_d; p.depth_pert = c->depth_pert;
  p.sn_ring = c->sn_ring; p.sm_ring = c->sm_ring;
  for (int k = 0; k < 3; ++k) {
    p.sn_sigma_white[k] = g.sn_sigma_white[k]; p.sn_sigma_rw[k] = g.sn_sigma_rw[k]; p.sn_bias[k] = g.sn_bias[k];
    p.sn_quant[k] = g.sn_quant[k]; p.sn_stuck_min[k] = g.sn_stuck_min[k]; p.sn_stuck_max[k] = g.sn_stuck_max[k];
  }
  p.dead_thr = c->dead_thr;
  p.pc_pts = c->pc_pts; p.pc_cell = c->pc_cell; p.pc_grid = c->pc_grid; p.pc_id = c->pc_id; p.pc_n = c->pc_n; p.pc_np = (c->pc_n + 15) / 16 * 16; p.tx_patch = c->tx_patch;
  p.pc_radius = g.pc_radius; p.pc_k = g.pc_k; p.pc_ks = g.pc_ks; p.pc_density = g.pc_density;
  p.sh_on = c->sh_on; p.sh_e = c->sh_e; p.pc_raw = c->pc_raw; p.sh_cnt = c->sh_cnt;
  p.rc_nodes = c->rc_nodes; p.rc_tri = c->rc_tri; p.rc_root = c->rc_root; p.rc_id = c->rc_id;
  p.shear_enable = (g.shear_enable && c->sh_on) ? 1 : 0; p.s_s = g.s_s; p.lambda_s = g.lambda_s; p.eta_enter = g.eta_enter; p.eta_exit = g.eta_exit;
}
}  // namespace

extern "C" {

const char* ts_version(void) { return "ts 0.1 (sm_100a)"; }

void ts_config_default(ts_config* c) {
  if (!c) return;
  std::memset(c, 0, sizeof(*c));
  c->n_envs = 1; c->n_links = 1; c->objs_per_env = 1;
  c->k_n = 500.f; c->c_n = 1.f; c->alpha = 1.2f; c->k_t = 2.f; c->k_omega = 2.f;  // Eq. 10
  c->mu = 1.0f;                                                                    // D2
  c->use_velocity = 1;
  c->eta_on = 5e-4f; c->eta_off = 5e-4f;
  c->s_d = 100.f; c->lambda_d = 8000.f; c->alpha_e = 1.2f; c->c_e = 1.f;
  c->r_prox = 0.020f; c->march_steps = 16;                                         // D1
  c->dt = 0.005f;
  c->tau = 0.05f; c->beta = 0.5f; c->alpha_load = 1.f; c->alpha_unload = 1.f;
  c->gain_min = 1.f; c->gain_max = 1.f;                                             // Eq. 27 off
  c->pc_radius = 0.01f; c->pc_k = 300.f; c->pc_ks = 10.f; c->pc_density = 100.f;    // A.6 P:267
  c->s_s = 100.f; c->lambda_s = 2000.f; c->eta_enter = 1e-5f; c->eta_exit = 1e-4f;  // A.7 P:304
  c->output_mask = TS_OUT_CONTACT | TS_OUT_DEPTH | TS_OUT_FT | TS_OUT_MARKER | TS_OUT_PROX;
}

const char* ts_last_error(const ts_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }
int32_t ts_n_taxels(const ts_ctx* ctx) { return ctx ? ctx->T : 0; }
int32_t ts_n_markers(const ts_ctx* ctx) { return ctx ? ctx->M : 0; }
int32_t ts_launches_per_step(const ts_ctx* ctx) {
  if (!ctx) return 0;
  return ((ctx->cfg.noise_enable && !ctx->fused) ? 3 : 2) +
         ((ctx->cfg.output_mask & (TS_OUT_DEPTH_NOISY | TS_OUT_PROX_NOISY | TS_OUT_MARKER_NOISY)) ? 1 : 0) +
         ((ctx->cfg.output_mask & TS_OUT_PROXPC) ? 1 : 0) + ((ctx->cfg.output_mask & (TS_OUT_DEPTH_RC | TS_OUT_NRM_RC)) ? 1 : 0) +
         ((ctx->cfg.shear_enable && (ctx->cfg.output_mask & (TS_OUT_MARKER | TS_OUT_MARKER_NOISY))) ? 1 : 0);
}

ts_status ts_create(const ts_config* cfg, int cuda_device, ts_ctx** out) {
  if (!cfg || !out) return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: NULL argument");
  *out = nullptr;
  const ts_layout* lay = cfg->layout;
  if (!lay || !lay->finalized) return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: layout missing or not finalised");
  if (cfg->n_envs < 1 || cfg->n_links < 1 || cfg->objs_per_env < 1)
    return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: n_envs, n_links, objs_per_env must be >= 1");
  if (!(cfg->eta_off <= cfg->eta_on)) return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: eta_off > eta_on");
  if (cfg->kernel_form < TS_FORM_AUTO || cfg->kernel_form > TS_FORM_SPLIT) return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: kernel_form");
  if (cfg->env_id_base < 0 || cfg->env_id_base + (int64_t)cfg->n_envs > (1LL << 32))
    return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: need 0 <= env_id_base and env_id_base + n_envs <= 2^32 (32-bit Philox counter word)");
  if (cfg->march_steps < 0 || cfg->march_steps > 64) return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: march_steps not in 0..64");
  if (!(cfg->alpha > 0.f) || !(cfg->r_prox >= 0.f) || !(cfg->lambda_d > 0.f) || !(cfg->c_e >= 0.f && cfg->c_e <= 1.f))
    return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: physics parameter out of range");
  if (cfg->noise_enable) {
    if (cfg->hyst_mode < TS_HYST_OFF || cfg->hyst_mode > TS_HYST_ASYM) return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: hyst_mode");
    if (!(cfg->p_dead >= 0.f && cfg->p_dead < 1.f)) return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: p_dead not in [0,1)");
    if (cfg->hyst_mode == TS_HYST_MAXWELL && !(cfg->tau > 0.f)) return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: tau <= 0");
    if (!(cfg->sigma_white_force >= 0.f) || !(cfg->sigma_white_torque >= 0.f) || !(cfg->quant_force >= 0.f) || !(cfg->quant_torque >= 0.f))
      return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: sigma_white / quant must be >= 0");
    if (!(cfg->xtalk_sigma >= 0.f) || std::ceil(3.0 * (double)cfg->xtalk_sigma) > 4.0)
      return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: xtalk_sigma not in [0, 4/3]");
    if (!(cfg->radius_noise >= 0.f) || !(cfg->radius_noise < INFINITY)) return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: radius_noise must be finite and >= 0");
    if (cfg->read_delay < 0 || cfg->read_jitter < 0 || cfg->read_delay + cfg->read_jitter > 64)
      return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: need 0 <= read_delay, read_jitter and read_delay + read_jitter <= 64");
    if ((long long)cfg->n_envs * 3LL * (cfg->read_delay + cfg->read_jitter) * ((lay->n_taxels + 31) / 32 * 32) >= (1LL << 32))
      return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: n_envs * n_taxels * (read_delay + read_jitter) too large (32-bit element indices)");
    if (!(cfg->gain_min > 0.f) || !(cfg->gain_min <= cfg->gain_max)) return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: need 0 < gain_min <= gain_max");
    if (!(cfg->stuck_min_force <= cfg->stuck_max_force) || !(cfg->stuck_min_torque <= cfg->stuck_max_torque))
      return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: stuck_min > stuck_max");
    for (int k = 0; k < 3; ++k)
      if (!(cfg->sn_sigma_white[k] >= 0.f) || !(cfg->sn_sigma_rw[k] >= 0.f) || !(cfg->sn_quant[k] >= 0.f) || !(cfg->sn_stuck_min[k] <= cfg->sn_stuck_max[k]))
        return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: sn_* knobs: sigma, quant >= 0 and stuck_min <= stuck_max");
    if ((cfg->output_mask & TS_OUT_MARKER_NOISY) && lay->marker_patch.empty())
      return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: marker_noisy requested but the layout has no markers");
  } else if (cfg->output_mask & (TS_OUT_FT_NOISY | TS_OUT_DEAD | TS_OUT_DEPTH_NOISY | TS_OUT_PROX_NOISY | TS_OUT_MARKER_NOISY)) {
    return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: noisy outputs and dead need noise_enable");
  }
  for (size_t t = 0; t < lay->link.size(); ++t)
    if (lay->link[t] >= cfg->n_links) return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: layout link index >= n_links");
  if ((long long)cfg->n_envs * 12LL * ((lay->n_taxels + 31) / 32 * 32) >= (1LL << 32))
    return fail(nullptr, TS_ERR_INVALID_ARG, "ts_create: n_envs * n_taxels too large (state uses 32-bit element indices)");

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev)
    return fail(nullptr, TS_ERR_CUDA, "ts_create: no such CUDA device");
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess) return fail(nullptr, TS_ERR_CUDA, "ts_create: cudaGetDeviceProperties");
  if (prop.major != 10) return fail(nullptr, TS_ERR_UNSUPPORTED, "ts_create: kernels are built for sm_100a only");

  ts_ctx* c = new (std::nothrow) ts_ctx();
  if (!c) return fail(nullptr, TS_ERR_OOM, "ts_create: host allocation");
  c->device = cuda_device;
  c->cfg = *cfg;
  c->cfg.layout = nullptr;
  DeviceGuard guard(cuda_device);

  // ---- layout -> device records; trailing filler slots are covered by filler patches ----
  const int T = lay->n_taxels;
  std::vector<float4> pos(T);
  std::vector<int32_t> meta(T, 0);
  for (int t = 0; t < T; ++t)
    pos[t] = make_float4(lay->pos[3 * t], lay->pos[3 * t + 1], lay->pos[3 * t + 2], lay->radius[t]);
  const int M = (int)lay->marker_patch.size();
  std::vector<TsPatch> pts;
  std::vector<double> tab;
  std::vector<double> tab8;   // [patch][4][8][8], zero-padded copies of the separable tables
  bool all_mma = true;        // every patch with markers fits the 8 x 8 DMMA tiles
  std::vector<int32_t> item1, item2(M > 0 ? M : 1, 0);
  int used = 0;
  for (size_t pi = 0; pi < lay->patch_start.size(); ++pi) {
    const ts_patch_desc& d = lay->desc[pi];
    TsPatch q{};
    q.start = lay->patch_start[pi]; q.nu = d.nu; q.nv = d.nv; q.n = d.nu * d.nv;
    q.link = d.link; q.mstart = lay->marker_start[pi]; q.mnu = d.marker_nu; q.mnv = d.marker_nv;
    q.eps = lay->patch_eps[pi];
    const double u[3] = {d.u_axis[0], d.u_axis[1], d.u_axis[2]}, v[3] = {d.v_axis[0], d.v_axis[1], d.v_axis[2]};
    q.ua = make_float4(d.u_axis[0], d.u_axis[1], d.u_axis[2], d.size_u);
    q.va = make_float4(d.v_axis[0], d.v_axis[1], d.v_axis[2], d.size_v);
    q.ctr = make_float4(d.origin[0], d.origin[1], d.origin[2], 0.f);
    q.na = make_float4(lay->nrm[3 * q.start], lay->nrm[3 * q.start + 1], lay->nrm[3 * q.start + 2], 0.f);  // = marker normal
    q.direct = (cfg->c_e != 1.0f || q.mnu * q.nv > TS_CHUNK) ? 1 : 0;
    q.tab = (int32_t)tab.size();
    q.i1off = (int32_t)item1.size();
    if (q.mnu > 0 && !q.direct) {
      // separable tables from the fp32 layout coordinates (the oracle's inputs), evaluated in double:
      // su(a,p) = u^.(x^m(a,0) - x(p,0)) / u^.u^,  GU = exp(-lambda su^2 u^.u^),  DU = su GU; same along v.
      const double lam = (double)cfg->lambda_d;
      const double uu = u[0] * u[0] + u[1] * u[1] + u[2] * u[2], vv = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
      auto coef = [&](int m, int t, const double* ax, double aa) {
        double s = 0.0;
        for (int k = 0; k < 3; ++k) s += ax[k] * ((double)lay->marker_pos[3 * m + k] - (double)lay->pos[3 * t + k]);
        return s / aa;
      };
      std::vector<double> GU(q.mnu * q.nu), DU(q.mnu * q.nu), GV(q.mnv * q.nv), DV(q.mnv * q.nv);
      for (int a = 0; a < q.mnu; ++a)
        for (int ip = 0; ip < q.nu; ++ip) {
          const double su = coef(q.mstart + a, q.start + ip, u, uu);
          GU[a * q.nu + ip] = std::exp(-lam * su * su * uu);
          DU[a * q.nu + ip] = su * GU[a * q.nu + ip];
        }
      for (int b = 0; b < q.mnv; ++b)
        for (int iq = 0; iq < q.nv; ++iq) {
          const double sv = coef(q.mstart + b * q.mnu, q.start + iq * q.nu, v, vv);
          GV[b * q.nv + iq] = std::exp(-lam * sv * sv * vv);
          DV[b * q.nv + iq] = sv * GV[b * q.nv + iq];
        }
      tab.insert(tab.end(), GU.begin(), GU.end());
      tab.insert(tab.end(), DU.begin(), DU.end());
      tab.insert(tab.end(), GV.begin(), GV.end());
      tab.insert(tab.end(), DV.begin(), DV.end());
      if (q.nu <= 8 && q.nv <= 8 && q.mnu <= 8 && q.mnv <= 8) {
        tab8.resize((pts.size() + 1) * 256, 0.0);
        double* t8 = tab8.data() + pts.size() * 256;
        for (int a = 0; a < q.mnu; ++a)
          for (int ip = 0; ip < q.nu; ++ip) { t8[a * 8 + ip] = GU[a * q.nu + ip]; t8[64 + a * 8 + ip] = DU[a * q.nu + ip]; }
        for (int b = 0; b < q.mnv; ++b)
          for (int iq = 0; iq < q.nv; ++iq) { t8[128 + b * 8 + iq] = GV[b * q.nv + iq]; t8[192 + b * 8 + iq] = DV[b * q.nv + iq]; }
      } else {
        all_mma = false;
      }
      for (int iq = 0; iq < q.nv; ++iq)
        for (int a = 0; a < q.mnu; ++a) item1.push_back(0);  // packed below, once the group-local index is known
    }
    if (q.mnu > 0 && q.direct) all_mma = false;
    pts.push_back(q);
    used = q.start + q.n;
  }
  for (int t = used; t < T; t += TS_BLOCK) {
    TsPatch q{};
    q.start = t; q.n = (T - t < TS_BLOCK) ? T - t : TS_BLOCK; q.nu = q.n; q.nv = 1; q.link = -1; q.mstart = M;
    q.tab = (int32_t)tab.size(); q.i1off = (int32_t)item1.size();
    q.ua = q.va = q.na = q.ctr = make_float4(0.f, 0.f, 0.f, 0.f);
    pts.push_back(q);
  }
  // ---- pack whole patches into groups of <= TS_BLOCK slots; markers of a group into chunks ----
  std::vector<TsGroup> groups;
  std::vector<TsChunk> chunks;
  int fpg = 1;
  for (size_t pi = 0; pi < pts.size();) {
    TsGroup g{};
    g.start = pts[pi].start; g.patch0 = (int32_t)pi; g.mstart = pts[pi].mstart; g.chunk0 = (int32_t)chunks.size();
    while (pi < pts.size() && g.count + pts[pi].n <= TS_BLOCK && g.npatch < TS_MAX_GROUP_PATCHES) {
      g.count += pts[pi].n; g.npatch += 1; g.mcount += pts[pi].mnu * pts[pi].mnv; ++pi;
    }
    if (g.npatch > fpg) fpg = g.npatch;
    for (int l = 0; l < g.npatch;) {  // chunks: pass-1 items and markers both fit one block
      TsChunk ck{};
      const TsPatch& f = pts[g.patch0 + l];
      ck.i1_begin = ck.i1_end = f.i1off; ck.m_begin = ck.m_end = f.mstart; ck.lp_begin = l;
      while (l < g.npatch) {
        const TsPatch& q = pts[g.patch0 + l];
        const int n1 = (q.mnu > 0 && !q.direct) ? q.mnu * q.nv : 0, nm = q.mnu * q.mnv;
        if (l > ck.lp_begin && ((ck.i1_end - ck.i1_begin) + n1 > TS_CHUNK || (ck.m_end - ck.m_begin) + nm > TS_CHUNK)) break;
        ck.i1_end += n1; ck.m_end += nm; ++l;
      }
      ck.lp_end = l;
      if (ck.m_end > ck.m_begin) chunks.push_back(ck);
    }
    g.nchunk = (int32_t)chunks.size() - g.chunk0;
    for (int l = 0; l < g.npatch; ++l) {  // group-local patch index: per taxel (in nrm.w) and per marker item
      const TsPatch& q = pts[g.patch0 + l];
      for (int t = q.start; t < q.start + q.n; ++t) {  // per-taxel word: patch index, grid width, neighbour bits
        int m = l | ((q.nu & 255) << 8);
        for (int a = 0; a < 4; ++a)
          if (lay->nbr[4 * t + a] >= 0) m |= 1 << (16 + a);
        meta[t] = m;
      }
      if (q.mnu > 0 && !q.direct)
        for (int iq = 0; iq < q.nv; ++iq)
          for (int a = 0; a < q.mnu; ++a) item1[q.i1off + iq * q.mnu + a] = l | (a << 8) | (iq << 16);
      for (int b = 0; b < q.mnv; ++b)
        for (int a = 0; a < q.mnu; ++a) item2[q.mstart + b * q.mnu + a] = l | (a << 8) | (b << 16);
    }
    groups.push_back(g);
  }
  std::vector<int32_t> glink(groups.size() * TS_MAX_GROUP_PATCHES, -1);
  for (size_t gi = 0; gi < groups.size(); ++gi)
    for (int l = 0; l < groups[gi].npatch; ++l) glink[gi * TS_MAX_GROUP_PATCHES + l] = pts[groups[gi].patch0 + l].link;
  c->h_groups = groups; c->h_glink = glink;
  if (item1.empty()) item1.push_back(0);
  if (tab.empty()) tab.push_back(0.0);
  tab8.resize(pts.size() * 256, 0.0);
  c->mk_mma = all_mma && M > 0;
  if (chunks.empty()) chunks.push_back(TsChunk{});
  std::vector<float4> mpos(M > 0 ? M : 1), mnrm(M > 0 ? M : 1);
  for (int j = 0; j < M; ++j) {
    // w = 1: the marker's patch is active (not removed by the link filter); read by the noisy marker readout (R10)
    mpos[j] = make_float4(lay->marker_pos[3 * j], lay->marker_pos[3 * j + 1], lay->marker_pos[3 * j + 2],
                          lay->radius[lay->patch_start[lay->marker_patch[j]]] > 0.f ? 1.f : 0.f);
    mnrm[j] = make_float4(lay->marker_nrm[3 * j], lay->marker_nrm[3 * j + 1], lay->marker_nrm[3 * j + 2], 0.f);
  }
  c->T = T; c->P = (int)pts.size(); c->M = M; c->G = (int)groups.size(); c->Tp = (T + 31) / 32 * 32;
  c->frames_per_group = fpg;
  c->nh = !cfg->noise_enable ? 0 : (cfg->hyst_mode == TS_HYST_MAXWELL ? 12 : (cfg->hyst_mode == TS_HYST_ASYM ? 6 : 0));
  c->dead_thr = (uint32_t)std::floor((double)cfg->p_dead * 4294967296.0);
  {
    TsStepParams sp;
    fill_params(c, sp);
    const unsigned long long smem = ts_step_smem_bytes(sp);
    if (smem > 200 * 1024) { delete c; return fail(nullptr, TS_ERR_UNSUPPORTED, "ts_create: objs_per_env too large for the shared-memory frames"); }
    const cudaError_t ea = (cudaError_t)ts_prepare_kernels(cuda_device, (int)smem);
    if (ea != cudaSuccess) { ts_status s_ = cuda_fail(nullptr, ea, "cudaFuncSetAttribute"); delete c; return s_; }
  }

  const size_t E = (size_t)cfg->n_envs, EK = E * cfg->objs_per_env;
#define TS_ALLOC(ptr, bytes)                                                          \
  do {                                                                                \
    cudaError_t e_ = cudaMalloc((void**)&(ptr), (bytes));                             \
    if (e_ != cudaSuccess) { ts_status s_ = cuda_fail(nullptr, e_, "cudaMalloc " #ptr); free_all(c); delete c; return s_; } \
  } while (0)
  TS_ALLOC(c->tx_pos, sizeof(float4) * T);
  TS_ALLOC(c->tx_meta, sizeof(int32_t) * T);
  TS_ALLOC(c->tx_patch, sizeof(int32_t) * T);
  TS_ALLOC(c->mk_pos, sizeof(float4) * mpos.size());
  TS_ALLOC(c->mk_nrm, sizeof(float4) * mnrm.size());
  TS_ALLOC(c->patches, sizeof(TsPatch) * pts.size());
  TS_ALLOC(c->groups, sizeof(TsGroup) * groups.size());
  TS_ALLOC(c->chunks, sizeof(TsChunk) * chunks.size());
  TS_ALLOC(c->grp_link, sizeof(int32_t) * glink.size());
  TS_ALLOC(c->mk_item1, sizeof(int32_t) * item1.size());
  TS_ALLOC(c->mk_item2, sizeof(int32_t) * item2.size());
  TS_ALLOC(c->mk_tab, sizeof(double) * tab.size());
  TS_ALLOC(c->mk_tab8, sizeof(double) * tab8.size());
  TS_ALLOC(c->g_type, sizeof(int32_t) * EK);
  TS_ALLOC(c->g_params, sizeof(float4) * EK);
  TS_ALLOC(c->env_perm, sizeof(int32_t) * E);
  TS_ALLOC(c->frames_g, (size_t)ts_frame_bytes() * E * pts.size() * cfg->objs_per_env);
  TS_ALLOC(c->patch_link, sizeof(int32_t) * pts.size());
  TS_ALLOC(c->st_flags, E * T);
  TS_ALLOC(c->reset_step, sizeof(uint32_t) * E);
  TS_ALLOC(c->episode, sizeof(uint32_t) * E);
  // Default (TS_FORM_AUTO): one fused launch.  (In round 1 the fused variant that carries the optional A.8 knobs ran past
  // the instruction-cache knee and AUTO chose two kernels for it; since the frames kernel and the DMMA marker path took
  // ~8 KB of SASS out of the step kernel the fused form wins with every knob set: DESIGN.md section 5.)
  c->fused = cfg->kernel_form == TS_FORM_FUSED ? true : (cfg->kernel_form == TS_FORM_SPLIT ? false : !TS_DEFAULT_SPLIT);
  if (cfg->noise_enable && !c->fused && !(cfg->output_mask & TS_OUT_FT)) TS_ALLOC(c->ft_scratch, sizeof(float) * E * T * 6);
  if (cfg->noise_enable && !c->fused && cfg->radius_noise != 0.f) TS_ALLOC(c->ft_scratch_r, sizeof(float) * E * T * 6);
  if (cfg->output_mask & (TS_OUT_DEPTH_NOISY | TS_OUT_PROX_NOISY)) {
    TS_ALLOC(c->sn_h, sizeof(float4) * E * T);
    TS_ALLOC(c->sn_d, sizeof(float2) * E * T);
    if ((cfg->output_mask & TS_OUT_DEPTH_NOISY) && cfg->radius_noise != 0.f) TS_ALLOC(c->depth_pert, sizeof(float) * E * T);
    if ((cfg->output_mask & TS_OUT_DEPTH_NOISY) && !(cfg->output_mask & TS_OUT_DEPTH)) TS_ALLOC(c->sc_depth, sizeof(float) * E * T);
    if ((cfg->output_mask & TS_OUT_PROX_NOISY) && !(cfg->output_mask & TS_OUT_PROX)) TS_ALLOC(c->sc_prox, sizeof(float) * E * T);
  }
  if (cfg->output_mask & TS_OUT_MARKER_NOISY) {
    TS_ALLOC(c->sm_h, sizeof(float) * E * M * 6);
    TS_ALLOC(c->sm_d, sizeof(float) * E * M * 3);
    if (!(cfg->output_mask & TS_OUT_MARKER)) TS_ALLOC(c->sc_marker, sizeof(float) * E * M * 3);
  }
  if (cfg->noise_enable && cfg->read_delay + cfg->read_jitter > 0) {   // Eq. 25 read delay of the scalar readouts (R10)
    const size_t S = (size_t)(cfg->read_delay + cfg->read_jitter);
    if (cfg->output_mask & (TS_OUT_DEPTH_NOISY | TS_OUT_PROX_NOISY)) {
      TS_ALLOC(c->sn_ring, sizeof(float2) * E * S * T);
      if (cudaMemset(c->sn_ring, 0, sizeof(float2) * E * S * T) != cudaSuccess) { free_all(c); delete c; return fail(nullptr, TS_ERR_CUDA, "ts_create: cudaMemset ring"); }
    }
    if ((cfg->output_mask & TS_OUT_MARKER_NOISY) && M > 0) {
      TS_ALLOC(c->sm_ring, sizeof(float) * E * S * M * 3);
      if (cudaMemset(c->sm_ring, 0, sizeof(float) * E * S * M * 3) != cudaSuccess) { free_all(c); delete c; return fail(nullptr, TS_ERR_CUDA, "ts_create: cudaMemset ring"); }
    }
  }
  if (cfg->noise_enable) {
    if (c->nh) TS_ALLOC(c->st_hyst, sizeof(float) * E * c->nh * c->Tp);
    TS_ALLOC(c->st_drift, sizeof(float) * E * 6 * c->Tp);
    // A slot is only read for a step of the current episode (ts_kernels.cu, noise_chain), i.e. after it was written;
    // the ring is zeroed once anyway so that no read can ever see uninitialised memory.
    if (cfg->read_delay + cfg->read_jitter > 0) {
      const size_t rb = sizeof(float) * E * 6 * c->Tp * (size_t)(cfg->read_delay + cfg->read_jitter);
      TS_ALLOC(c->st_ring, rb);
      if (cudaMemset(c->st_ring, 0, rb) != cudaSuccess) { free_all(c); delete c; return fail(nullptr, TS_ERR_CUDA, "ts_create: cudaMemset ring"); }
    }
  }
#undef TS_ALLOC
  cudaError_t e = cudaSuccess;
  auto cp = [&](void* d, const void* h, size_t b) { if (e == cudaSuccess) e = cudaMemcpy(d, h, b, cudaMemcpyHostToDevice); };
  cp(c->tx_pos, pos.data(), sizeof(float4) * T);
  cp(c->tx_meta, meta.data(), sizeof(int32_t) * T);
  {
    std::vector<int32_t> tpatch(T, 0);
    for (size_t pi = 0; pi < pts.size(); ++pi)
      for (int t = pts[pi].start; t < pts[pi].start + pts[pi].n && t < T; ++t) tpatch[t] = (int32_t)pi;
    cp(c->tx_patch, tpatch.data(), sizeof(int32_t) * T);
  }
  cp(c->mk_pos, mpos.data(), sizeof(float4) * mpos.size());
  cp(c->mk_nrm, mnrm.data(), sizeof(float4) * mnrm.size());
  cp(c->patches, pts.data(), sizeof(TsPatch) * pts.size());
  cp(c->groups, groups.data(), sizeof(TsGroup) * groups.size());
  cp(c->chunks, chunks.data(), sizeof(TsChunk) * chunks.size());
  cp(c->grp_link, glink.data(), sizeof(int32_t) * glink.size());
  {
    std::vector<int32_t> plink(pts.size());
    for (size_t pi = 0; pi < pts.size(); ++pi) plink[pi] = pts[pi].link;
    cp(c->patch_link, plink.data(), sizeof(int32_t) * plink.size());
  }
  cp(c->mk_item1, item1.data(), sizeof(int32_t) * item1.size());
  cp(c->mk_item2, item2.data(), sizeof(int32_t) * item2.size());
  cp(c->mk_tab, tab.data(), sizeof(double) * tab.size());
  cp(c->mk_tab8, tab8.data(), sizeof(double) * tab8.size());
  if (e == cudaSuccess) e = cudaMemset(c->g_type, 0, sizeof(int32_t) * EK);
  if (e == cudaSuccess) e = cudaMemset(c->g_params, 0, sizeof(float4) * EK);
  if (e == cudaSuccess) e = cudaMemset(c->reset_step, 0, sizeof(uint32_t) * E);
  if (e == cudaSuccess) e = cudaMemset(c->episode, 0, sizeof(uint32_t) * E);
  if (e == cudaSuccess) {  // episode 0: zero state, draw the dead mask
    TsStepParams p;
    fill_params(c, p);
    e = (cudaError_t)ts_launch_reset_state(p, nullptr, c->dead_thr, c->nh, nullptr);
    if (e == cudaSuccess && (c->sn_d || c->sm_d)) e = (cudaError_t)ts_launch_reset_scalar(p, nullptr, nullptr);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
  }
  if (e != cudaSuccess) { ts_status s = cuda_fail(nullptr, e, "ts_create: upload"); free_all(c); delete c; return s; }
  *out = c;
  return TS_OK;
}

ts_status ts_set_geometry(ts_ctx* c, const ts_geometry* geo, void* stream) {
  if (!c) return TS_ERR_INVALID_ARG;
  if (!geo || !geo->type || !geo->params) return fail(c, TS_ERR_INVALID_ARG, "ts_set_geometry: NULL argument");
  const int E = c->cfg.n_envs, K = c->cfg.objs_per_env;
  const size_t EK = (size_t)E * K;
  if (geo->n_grids < 0 || (geo->n_grids > 0 && (!geo->grids || geo->grid_n < 2 || geo->grid_n > 512 || !(geo->voxel > 0.f))))
    return fail(c, TS_ERR_INVALID_ARG, "ts_set_geometry: bad grid bank");
  for (size_t i = 0; i < EK; ++i) {
    const int t = geo->type[i];
    if (t < TS_GEOM_NONE || t > TS_GEOM_SDF) return fail(c, TS_ERR_INVALID_ARG, "ts_set_geometry: unknown type");
    if (t == TS_GEOM_SDF) {
      const float id = geo->params[4 * i];
      if (!(id >= 0.f) || id >= (float)geo->n_grids || id != std::floor(id)) return fail(c, TS_ERR_INVALID_ARG, "ts_set_geometry: grid id out of range");
    }
  }
  const int N = geo->grid_n;
  if (geo->n_grids > 0 && ts_bank_elems_per_grid(N) * (unsigned long long)geo->n_grids >= (1ULL << 31))
    return fail(c, TS_ERR_UNSUPPORTED, "ts_set_geometry: bank larger than 2^31 cells (32-bit cell indices)");
  DeviceGuard guard(c->device);
  cudaStream_t st = (cudaStream_t)stream;
  // From here on the old geometry is gone: every failure path leaves the ctx WITHOUT geometry (ts_step refuses), never
  // with new descriptors next to an old or missing bank.  Allocation first, uploads last.
  c->have_geometry = false;
  c->n_grids = 0;
  size_t lin = 0;
  if (geo->n_grids > 0) {
    const size_t need = sizeof(float4) * ts_bank_elems_per_grid(N) * geo->n_grids;
    lin = sizeof(float) * (size_t)N * N * N * geo->n_grids;
    if (need > c->bank_bytes || lin > c->bank_stage_bytes) TS_CUDA(c, cudaStreamSynchronize(st));  // steps in flight still read them
    if (need > c->bank_bytes) {
      cudaFree(c->bank); c->bank = nullptr; c->bank_bytes = 0;
      TS_CUDA(c, cudaMalloc((void**)&c->bank, need));
      c->bank_bytes = need;
    }
    if (lin > c->bank_stage_bytes) {  // linear staging copy of the bank, kept for the next call
      cudaFree(c->bank_stage); c->bank_stage = nullptr; c->bank_stage_bytes = 0;
      TS_CUDA(c, cudaMalloc((void**)&c->bank_stage, lin));
      c->bank_stage_bytes = lin;
    }
  }
  // Block -> env order of the step kernel: envs sorted (stably) by the geometry of their first object -- type, then
  // grid id -- so that the ~740 blocks resident at any time gather from one grid of the bank (it stays in L2: 8 x 96^3
  // quad-layout grids are 113 MB, one is 14 MB) and run the same march loop.  Scheduling only: results do not depend on it.
  c->h_perm.resize(E);
  for (int e = 0; e < E; ++e) c->h_perm[e] = e;
  auto key = [&](int e) {
    const int t = geo->type[(size_t)e * K];
    return t * 4096 + (t == TS_GEOM_SDF ? (int)geo->params[4 * (size_t)e * K] % 4096 : 0);
  };
  std::stable_sort(c->h_perm.begin(), c->h_perm.end(), [&](int a, int b) { return key(a) < key(b); });
  TS_CUDA(c, cudaMemcpyAsync(c->env_perm, c->h_perm.data(), sizeof(int32_t) * E, cudaMemcpyHostToDevice, st));
  TS_CUDA(c, cudaMemcpyAsync(c->g_type, geo->type, sizeof(int32_t) * EK, cudaMemcpyHostToDevice, st));
  TS_CUDA(c, cudaMemcpyAsync(c->g_params, geo->params, sizeof(float4) * EK, cudaMemcpyHostToDevice, st));
  if (geo->n_grids > 0) {
    TS_CUDA(c, cudaMemcpyAsync(c->bank_stage, geo->grids, lin, cudaMemcpyHostToDevice, st));
    const cudaError_t e = (cudaError_t)ts_launch_retile(c->bank_stage, c->bank, geo->n_grids, N, st);
    if (e != cudaSuccess) return cuda_fail(c, e, "ts_set_geometry: retile launch");
  }
  TS_CUDA(c, cudaStreamSynchronize(st));  // the caller may free or reuse its arrays once this returns
  if (geo->n_grids > 0) { c->grid_n = N; c->voxel = geo->voxel; c->n_grids = geo->n_grids; }
  c->have_geometry = true;
  return TS_OK;
}

namespace {
// median-split BVH over the triangles tri[lo, hi) of one mesh (indices into `order`); returns the node index
struct BvhBuild {
  const float* V;             // vertices of the mesh
  const int32_t* T;           // triangles of the mesh (local vertex indices)
  std::vector<int32_t> order; // triangle permutation (leaf order)
  std::vector<float4>* nodes; // flattened nodes (2 float4 each), shared by all meshes
  std::vector<float4>* tris;  // leaf-ordered triangles (3 float4 each), shared by all meshes
  void box(int t, float lo[3], float hi[3]) const {
    for (int a = 0; a < 3; ++a) { lo[a] = INFINITY; hi[a] = -INFINITY; }
    for (int v = 0; v < 3; ++v)
      for (int a = 0; a < 3; ++a) { const float x = V[3 * T[3 * t + v] + a]; lo[a] = std::fmin(lo[a], x); hi[a] = std::fmax(hi[a], x); }
  }
  int build(int lo_i, int hi_i) {
    float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (int i = lo_i; i < hi_i; ++i) {
      float l[3], h[3];
      box(order[i], l, h);
      for (int a = 0; a < 3; ++a) { lo[a] = std::fmin(lo[a], l[a]); hi[a] = std::fmax(hi[a], h[a]); }
    }
    const int node = (int)(nodes->size() / 2);
    nodes->push_back(make_float4(lo[0], lo[1], lo[2], 0.f));
    nodes->push_back(make_float4(hi[0], hi[1], hi[2], 0.f));
    auto seti = [&](size_t idx, int v) { int32_t iv = v; std::memcpy(&(*nodes)[idx].w, &iv, 4); };
    if (hi_i - lo_i <= 4) {   // leaf: triangles appended in leaf order
      seti((size_t)2 * node, (int)(tris->size() / 3));
      seti((size_t)2 * node + 1, hi_i - lo_i);
      for (int i = lo_i; i < hi_i; ++i)
        for (int v = 0; v < 3; ++v) { const float* p = V + 3 * T[3 * order[i] + v]; tris->push_back(make_float4(p[0], p[1], p[2], 0.f)); }
      return node;
    }
    int ax = 0;
    if (hi[1] - lo[1] > hi[ax] - lo[ax]) ax = 1;
    if (hi[2] - lo[2] > hi[ax] - lo[ax]) ax = 2;
    const int mid = (lo_i + hi_i) / 2;
    std::nth_element(order.begin() + lo_i, order.begin() + mid, order.begin() + hi_i, [&](int a, int b) {
      float la[3], ha[3], lb[3], hb[3];
      box(a, la, ha); box(b, lb, hb);
      return la[ax] + ha[ax] < lb[ax] + hb[ax];
    });
    const int left = build(lo_i, mid), right = build(mid, hi_i);
    seti((size_t)2 * node, left);
    seti((size_t)2 * node + 1, -right);
    return node;
  }
};
}  // namespace

ts_status ts_set_meshes(ts_ctx* c, const ts_meshes* m, void* stream) {
  if (!c) return TS_ERR_INVALID_ARG;
  if (!m || m->n_meshes < 1 || !m->vert_off || !m->tri_off || !m->verts || !m->tris || !m->mesh_id)
    return fail(c, TS_ERR_INVALID_ARG, "ts_set_meshes: NULL argument or empty bank");
  const int G = m->n_meshes;
  const size_t EK = (size_t)c->cfg.n_envs * c->cfg.objs_per_env;
  for (size_t i = 0; i < EK; ++i)
    if (m->mesh_id[i] >= G) return fail(c, TS_ERR_INVALID_ARG, "ts_set_meshes: mesh id out of range");
  std::vector<float4> nodes, tris;
  std::vector<int32_t> roots(G);
  for (int g = 0; g < G; ++g) {
    const int nv = m->vert_off[g + 1] - m->vert_off[g], nt = m->tri_off[g + 1] - m->tri_off[g];
    if (nv < 3 || nt < 1) return fail(c, TS_ERR_INVALID_ARG, "ts_set_meshes: empty mesh");
    const int32_t* T = m->tris + (size_t)m->tri_off[g] * 3;
    for (int i = 0; i < 3 * nt; ++i)
      if (T[i] < 0 || T[i] >= nv) return fail(c, TS_ERR_INVALID_ARG, "ts_set_meshes: vertex index out of range");
    BvhBuild b;
    b.V = m->verts + (size_t)m->vert_off[g] * 3; b.T = T; b.nodes = &nodes; b.tris = &tris;
    b.order.resize(nt);
    for (int i = 0; i < nt; ++i) b.order[i] = i;
    roots[g] = b.build(0, nt);
  }
  DeviceGuard guard(c->device);
  cudaStream_t st = (cudaStream_t)stream;
  c->have_mesh = false;
  TS_CUDA(c, cudaStreamSynchronize(st));
  cudaFree(c->rc_nodes); cudaFree(c->rc_tri); cudaFree(c->rc_root); cudaFree(c->rc_id);
  c->rc_nodes = nullptr; c->rc_tri = nullptr; c->rc_root = nullptr; c->rc_id = nullptr;
  TS_CUDA(c, cudaMalloc((void**)&c->rc_nodes, sizeof(float4) * nodes.size()));
  TS_CUDA(c, cudaMalloc((void**)&c->rc_tri, sizeof(float4) * tris.size()));
  TS_CUDA(c, cudaMalloc((void**)&c->rc_root, sizeof(int32_t) * G));
  TS_CUDA(c, cudaMalloc((void**)&c->rc_id, sizeof(int32_t) * EK));
  TS_CUDA(c, cudaMemcpyAsync(c->rc_nodes, nodes.data(), sizeof(float4) * nodes.size(), cudaMemcpyHostToDevice, st));
  TS_CUDA(c, cudaMemcpyAsync(c->rc_tri, tris.data(), sizeof(float4) * tris.size(), cudaMemcpyHostToDevice, st));
  TS_CUDA(c, cudaMemcpyAsync(c->rc_root, roots.data(), sizeof(int32_t) * G, cudaMemcpyHostToDevice, st));
  TS_CUDA(c, cudaMemcpyAsync(c->rc_id, m->mesh_id, sizeof(int32_t) * EK, cudaMemcpyHostToDevice, st));
  TS_CUDA(c, cudaStreamSynchronize(st));
  c->have_mesh = true;
  return TS_OK;
}

ts_status ts_set_pointclouds(ts_ctx* c, const ts_pointclouds* pc, void* stream) {
  if (!c) return TS_ERR_INVALID_ARG;
  if (!pc || !pc->points || !pc->cloud_id || pc->n_clouds < 1 || pc->n_points < 1)
    return fail(c, TS_ERR_INVALID_ARG, "ts_set_pointclouds: NULL argument or empty bank");
  if (!(c->cfg.pc_radius > 0.f)) return fail(c, TS_ERR_INVALID_ARG, "ts_set_pointclouds: pc_radius must be > 0");
  const int G = pc->n_clouds, N = pc->n_points;
  const size_t EK = (size_t)c->cfg.n_envs * c->cfg.objs_per_env;
  for (size_t i = 0; i < EK; ++i)
    if (pc->cloud_id[i] >= G) return fail(c, TS_ERR_INVALID_ARG, "ts_set_pointclouds: cloud id out of range");
  if ((long long)G * N >= (1LL << 31)) return fail(c, TS_ERR_UNSUPPORTED, "ts_set_pointclouds: bank larger than 2^31 points");
  // static spatial index ("organized in a static BVH"): per cloud a uniform grid with cell = sensing radius / TS_PC_REACH,
  // points counting-sorted by linear cell index (x fastest), cell_start[ncell + 1]
  const float cell = c->cfg.pc_radius / (float)TS_PC_REACH;
  std::vector<TsPcGrid> grids(G);
  std::vector<int32_t> cells;
  std::vector<float4> sorted((size_t)G * N);
  for (int g = 0; g < G; ++g) {
    const float* P = pc->points + (size_t)g * N * 3;
    float lo[3] = {P[0], P[1], P[2]}, hi[3] = {P[0], P[1], P[2]};
    for (int i = 0; i < N; ++i)
      for (int a = 0; a < 3; ++a) {
        if (!std::isfinite(P[3 * i + a])) return fail(c, TS_ERR_INVALID_ARG, "ts_set_pointclouds: non-finite point");
        lo[a] = std::fmin(lo[a], P[3 * i + a]); hi[a] = std::fmax(hi[a], P[3 * i + a]);
      }
    TsPcGrid& gr = grids[g];
    gr.ox = lo[0]; gr.oy = lo[1]; gr.oz = lo[2]; gr.inv_cell = 1.0f / cell;
    gr.nx = (int)std::floor((hi[0] - lo[0]) * gr.inv_cell) + 1; gr.ny = (int)std::floor((hi[1] - lo[1]) * gr.inv_cell) + 1;
    gr.nz = (int)std::floor((hi[2] - lo[2]) * gr.inv_cell) + 1;
    const long long ncell = (long long)gr.nx * gr.ny * gr.nz;
    if (ncell > (1LL << 26)) return fail(c, TS_ERR_UNSUPPORTED, "ts_set_pointclouds: cloud extent / pc_radius too large for the grid");
    gr.cell0 = (int32_t)cells.size(); gr.pt0 = g * N;
    std::vector<int32_t> cidx(N), start((size_t)ncell + 1, 0);
    for (int i = 0; i < N; ++i) {
      // the same fp32 expression the kernel uses for the taxel's cell
      int ci = (int)std::floor((P[3 * i] - gr.ox) * gr.inv_cell), cj = (int)std::floor((P[3 * i + 1] - gr.oy) * gr.inv_cell),
          ck = (int)std::floor((P[3 * i + 2] - gr.oz) * gr.inv_cell);
      ci = std::min(std::max(ci, 0), gr.nx - 1); cj = std::min(std::max(cj, 0), gr.ny - 1); ck = std::min(std::max(ck, 0), gr.nz - 1);
      cidx[i] = (ck * gr.ny + cj) * gr.nx + ci;
      start[(size_t)cidx[i] + 1] += 1;
    }
    for (long long k = 0; k < ncell; ++k) start[k + 1] += start[k];
    std::vector<int32_t> fill(start.begin(), start.end() - 1);
    for (int i = 0; i < N; ++i) {   // .w carries the point's index in the caller's order (the shear anchors are indexed by it)
      float wi;
      std::memcpy(&wi, &i, sizeof(float));
      sorted[(size_t)g * N + fill[cidx[i]]++] = make_float4(P[3 * i], P[3 * i + 1], P[3 * i + 2], wi);
    }
    cells.insert(cells.end(), start.begin(), start.end());
  }
  DeviceGuard guard(c->device);
  cudaStream_t st = (cudaStream_t)stream;
  c->have_pc = false;
  TS_CUDA(c, cudaStreamSynchronize(st));   // steps in flight may still read the old index
  cudaFree(c->sh_on); cudaFree(c->sh_e); cudaFree(c->pc_raw); cudaFree(c->sh_cnt);
  c->sh_on = nullptr; c->sh_e = nullptr; c->pc_raw = nullptr; c->sh_cnt = nullptr;
  cudaFree(c->pc_pts); cudaFree(c->pc_cell); cudaFree(c->pc_grid); cudaFree(c->pc_id);
  c->pc_pts = nullptr; c->pc_cell = nullptr; c->pc_grid = nullptr; c->pc_id = nullptr;
  TS_CUDA(c, cudaMalloc((void**)&c->pc_pts, sizeof(float4) * sorted.size()));
  TS_CUDA(c, cudaMalloc((void**)&c->pc_cell, sizeof(int32_t) * cells.size()));
  TS_CUDA(c, cudaMalloc((void**)&c->pc_grid, sizeof(TsPcGrid) * G));
  TS_CUDA(c, cudaMalloc((void**)&c->pc_id, sizeof(int32_t) * EK));
  TS_CUDA(c, cudaMemcpyAsync(c->pc_pts, sorted.data(), sizeof(float4) * sorted.size(), cudaMemcpyHostToDevice, st));
  TS_CUDA(c, cudaMemcpyAsync(c->pc_cell, cells.data(), sizeof(int32_t) * cells.size(), cudaMemcpyHostToDevice, st));
  TS_CUDA(c, cudaMemcpyAsync(c->pc_grid, grids.data(), sizeof(TsPcGrid) * G, cudaMemcpyHostToDevice, st));
  TS_CUDA(c, cudaMemcpyAsync(c->pc_id, pc->cloud_id, sizeof(int32_t) * EK, cudaMemcpyHostToDevice, st));
  if (c->cfg.shear_enable && c->M > 0) {   // Eq. 22 anchors: one per (env, patch, object, tracked point)
    const size_t ns = (size_t)c->cfg.n_envs * c->P * c->cfg.objs_per_env * (size_t)((N + 15) / 16 * 16);
    std::vector<float4> raw((size_t)G * N);
    for (size_t i = 0; i < raw.size(); ++i) raw[i] = make_float4(pc->points[3 * i], pc->points[3 * i + 1], pc->points[3 * i + 2], 0.f);
    TS_CUDA(c, cudaMalloc((void**)&c->sh_on, ns));
    TS_CUDA(c, cudaMalloc((void**)&c->sh_e, sizeof(float4) * ns));
    TS_CUDA(c, cudaMalloc((void**)&c->pc_raw, sizeof(float4) * raw.size()));
    TS_CUDA(c, cudaMemsetAsync(c->sh_on, 0, ns, st));
    const size_t ncnt = (size_t)c->cfg.n_envs * c->P * c->cfg.objs_per_env;
    TS_CUDA(c, cudaMalloc((void**)&c->sh_cnt, sizeof(int32_t) * ncnt));
    TS_CUDA(c, cudaMemsetAsync(c->sh_cnt, 0, sizeof(int32_t) * ncnt, st));
    TS_CUDA(c, cudaMemcpyAsync(c->pc_raw, raw.data(), sizeof(float4) * raw.size(), cudaMemcpyHostToDevice, st));
  }
  TS_CUDA(c, cudaStreamSynchronize(st));
  c->pc_n = N;
  c->have_pc = true;
  return TS_OK;
}

ts_status ts_step(ts_ctx* c, const ts_step_in* in, const ts_step_out* out, void* stream) {
  if (!c) return TS_ERR_INVALID_ARG;
  if (!in || !out) return fail(c, TS_ERR_INVALID_ARG, "ts_step: NULL argument");
  if (!c->have_geometry) return fail(c, TS_ERR_STATE, "ts_step before ts_set_geometry");
  if (!in->link_pos || !in->link_quat || !in->link_linvel || !in->link_angvel || !in->obj_pos || !in->obj_quat ||
      !in->obj_linvel || !in->obj_angvel)
    return fail(c, TS_ERR_INVALID_ARG, "ts_step: NULL input pointer");
  {  // output_mask contract (ts.h): bit set <=> pointer given
    const void* ptr[13] = {out->contact, out->depth, out->ft, out->marker, out->prox, out->ft_noisy, out->dead,
                           out->depth_noisy, out->prox_noisy, out->marker_noisy, out->proxpc, out->depth_rc, out->nrm_rc};
    for (int b = 0; b < 13; ++b) {
      const bool want = (c->cfg.output_mask >> b) & 1u;
      if (want && !ptr[b]) return fail(c, TS_ERR_INVALID_ARG, "ts_step: an output declared in output_mask is NULL");
      if (!want && ptr[b]) return fail(c, TS_ERR_INVALID_ARG, "ts_step: an output not declared in output_mask is non-NULL");
    }
  }
  if ((out->ft_noisy || out->dead) && !c->cfg.noise_enable) return fail(c, TS_ERR_INVALID_ARG, "ts_step: ft_noisy / dead need noise_enable");
  if (out->marker && c->M == 0) return fail(c, TS_ERR_INVALID_ARG, "ts_step: marker requested but the layout has no markers");
  const uintptr_t al = (uintptr_t)out->contact | (uintptr_t)out->depth | (uintptr_t)out->ft | (uintptr_t)out->marker |
                       (uintptr_t)out->prox | (uintptr_t)out->ft_noisy | (uintptr_t)out->dead | (uintptr_t)in->link_quat |
                       (uintptr_t)in->obj_quat;
  if (al & 15) return fail(c, TS_ERR_INVALID_ARG, "ts_step: pointers must be 16-byte aligned");
  DeviceGuard guard(c->device);
  TsStepParams p;
  fill_params(c, p);
  p.link_pos = in->link_pos; p.link_quat = in->link_quat; p.link_linvel = in->link_linvel; p.link_angvel = in->link_angvel;
  p.obj_pos = in->obj_pos; p.obj_quat = in->obj_quat; p.obj_linvel = in->obj_linvel; p.obj_angvel = in->obj_angvel;
  p.contact = out->contact; p.depth = out->depth; p.ft = out->ft; p.marker = out->marker; p.prox = out->prox;
  p.ft_noisy = out->ft_noisy; p.dead = out->dead;
  p.depth_noisy = out->depth_noisy; p.prox_noisy = out->prox_noisy; p.marker_noisy = out->marker_noisy;
  p.depth_rc = out->depth_rc; p.nrm_rc = out->nrm_rc;
  if ((p.depth_rc || p.nrm_rc) && !c->have_mesh) return fail(c, TS_ERR_STATE, "ts_step: raycast outputs requested before ts_set_meshes");
  p.proxpc = out->proxpc;
  if (p.proxpc && !c->have_pc) return fail(c, TS_ERR_STATE, "ts_step: proxpc requested before ts_set_pointclouds");
  const bool scalar_noisy = p.depth_noisy || p.prox_noisy || p.marker_noisy;
  if (p.depth_noisy && !p.depth) p.depth = c->sc_depth;      // clean inputs of the noisy readouts the caller did not ask for
  if (p.prox_noisy && !p.prox) p.prox = c->sc_prox;
  if (p.marker_noisy && !p.marker) p.marker = c->sc_marker;
  if (!p.depth_noisy) p.depth_pert = nullptr;
  cudaStream_t st = (cudaStream_t)stream;
  const bool split = c->cfg.noise_enable && !c->fused;
  if (split && !p.ft) {
    if (!c->ft_scratch) return fail(c, TS_ERR_INVALID_ARG, "ts_step: ft is NULL although TS_OUT_FT is set in output_mask");
    p.ft = c->ft_scratch;
  }
  const bool rec = c->timing && c->ev_used + 4 <= c->ev.size();   // pool exhausted: later steps are not recorded
  cudaEvent_t* ev = rec ? &c->ev[c->ev_used] : nullptr;
  if (rec) { p.clock = c->clock_buf + 2 * (c->ev_used / 4); c->ev_used += 4; TS_CUDA(c, cudaEventRecord(ev[0], st)); }
  cudaError_t e = (cudaError_t)ts_launch_frames(p, st);
  if (e != cudaSuccess) return cuda_fail(c, e, "ts_step: frames launch");
  if (rec && c->timing_detail) TS_CUDA(c, cudaEventRecord(ev[1], st));
  e = (cudaError_t)ts_launch_step(p, c->fused ? 1 : 0, st);
  if (e != cudaSuccess) return cuda_fail(c, e, "ts_step: launch");
  if (rec && c->timing_detail) TS_CUDA(c, cudaEventRecord(ev[2], st));
  if (split) {
    e = (cudaError_t)ts_launch_noise(p, st);
    if (e != cudaSuccess) return cuda_fail(c, e, "ts_step: noise launch");
  }
  if (c->cfg.shear_enable && p.marker) {
    if (!c->sh_on) return fail(c, TS_ERR_STATE, "ts_step: shear_enable needs ts_set_pointclouds before the first step");
    e = (cudaError_t)ts_launch_shear(p, st);
    if (e != cudaSuccess) return cuda_fail(c, e, "ts_step: shear launch");
  }
  if (p.depth_rc || p.nrm_rc) {
    e = (cudaError_t)ts_launch_raycast(p, st);
    if (e != cudaSuccess) return cuda_fail(c, e, "ts_step: raycast launch");
  }
  if (p.proxpc) {
    e = (cudaError_t)ts_launch_proxpc(p, st);
    if (e != cudaSuccess) return cuda_fail(c, e, "ts_step: proxpc launch");
  }
  if (scalar_noisy) {
    e = (cudaError_t)ts_launch_scalar_noise(p, st);
    if (e != cudaSuccess) return cuda_fail(c, e, "ts_step: scalar noise launch");
  }
  if (rec) TS_CUDA(c, cudaEventRecord(ev[3], st));
  c->gstep += 1;
  return TS_OK;
}

ts_status ts_step_host(ts_ctx* c, const ts_step_in* in, const ts_step_out* out, void* stream) {
  if (!c) return TS_ERR_INVALID_ARG;
  if (!in || !out) return fail(c, TS_ERR_INVALID_ARG, "ts_step_host: NULL argument");
  DeviceGuard guard(c->device);
  cudaStream_t st = (cudaStream_t)stream;
  const size_t E = (size_t)c->cfg.n_envs, L = (size_t)c->cfg.n_links, K = (size_t)c->cfg.objs_per_env, T = (size_t)c->T;
  const float* hin[8] = {in->link_pos, in->link_quat, in->link_linvel, in->link_angvel,
                         in->obj_pos, in->obj_quat, in->obj_linvel, in->obj_angvel};
  const size_t in_bytes[8] = {E * L * 12, E * L * 16, E * L * 12, E * L * 12, E * K * 12, E * K * 16, E * K * 12, E * K * 12};
  void* hout[13] = {out->contact, out->depth, out->ft, out->marker, out->prox, out->ft_noisy, out->dead,
                    out->depth_noisy, out->prox_noisy, out->marker_noisy, out->proxpc, out->depth_rc, out->nrm_rc};
  const size_t out_bytes[13] = {E * T, E * T * 4, E * T * 24, E * (size_t)c->M * 12, E * T * 4, E * T * 24, E * T,
                                E * T * 4, E * T * 4, E * (size_t)c->M * 12, E * T * 24, E * T * 4, E * T * 12};
  for (int i = 0; i < 8; ++i) {
    if (!hin[i]) return fail(c, TS_ERR_INVALID_ARG, "ts_step_host: NULL input pointer");
    if (!c->stage_in[i]) TS_CUDA(c, cudaMalloc((void**)&c->stage_in[i], in_bytes[i]));
    TS_CUDA(c, cudaMemcpyAsync(c->stage_in[i], hin[i], in_bytes[i], cudaMemcpyHostToDevice, st));
  }
  for (int i = 0; i < 13; ++i)
    if (hout[i] && !c->stage_out[i]) TS_CUDA(c, cudaMalloc(&c->stage_out[i], out_bytes[i] ? out_bytes[i] : 16));
  ts_step_in din = {c->stage_in[0], c->stage_in[1], c->stage_in[2], c->stage_in[3],
                    c->stage_in[4], c->stage_in[5], c->stage_in[6], c->stage_in[7]};
  ts_step_out dout = {hout[0] ? (uint8_t*)c->stage_out[0] : nullptr, hout[1] ? (float*)c->stage_out[1] : nullptr,
                      hout[2] ? (float*)c->stage_out[2] : nullptr,   hout[3] ? (float*)c->stage_out[3] : nullptr,
                      hout[4] ? (float*)c->stage_out[4] : nullptr,   hout[5] ? (float*)c->stage_out[5] : nullptr,
                      hout[6] ? (uint8_t*)c->stage_out[6] : nullptr, hout[7] ? (float*)c->stage_out[7] : nullptr,
                      hout[8] ? (float*)c->stage_out[8] : nullptr,   hout[9] ? (float*)c->stage_out[9] : nullptr,
                      hout[10] ? (float*)c->stage_out[10] : nullptr, hout[11] ? (float*)c->stage_out[11] : nullptr,
                      hout[12] ? (float*)c->stage_out[12] : nullptr};
  const ts_status s = ts_step(c, &din, &dout, stream);
  if (s != TS_OK) return s;
  for (int i = 0; i < 13; ++i)
    if (hout[i]) TS_CUDA(c, cudaMemcpyAsync(hout[i], c->stage_out[i], out_bytes[i], cudaMemcpyDeviceToHost, st));
  return TS_OK;
}

ts_status ts_reset(ts_ctx* c, const uint8_t* env_mask_dev, void* stream) {
  if (!c) return TS_ERR_INVALID_ARG;
  DeviceGuard guard(c->device);
  TsStepParams p;
  fill_params(c, p);
  cudaError_t e = (cudaError_t)ts_launch_reset_counters(c->reset_step, c->episode, env_mask_dev, c->cfg.n_envs, c->gstep, stream);
  if (e == cudaSuccess) e = (cudaError_t)ts_launch_reset_state(p, env_mask_dev, c->dead_thr, c->nh, stream);
  if (e == cudaSuccess && (c->sn_d || c->sm_d)) e = (cudaError_t)ts_launch_reset_scalar(p, env_mask_dev, stream);
  if (e == cudaSuccess && c->sh_on) e = (cudaError_t)ts_launch_reset_shear(p, env_mask_dev, stream);
  if (e != cudaSuccess) return cuda_fail(c, e, "ts_reset: launch");
  return TS_OK;
}

// ---- allocation-free contact depth (include/ts.h) -----------------------------------------------------------------
ts_status ts_depth_static(int32_t n_envs, int32_t n_links, int32_t n_taxels, const float* taxel_pos, const float* taxel_radius,
                          const int32_t* taxel_link, const float* link_pos, const float* link_quat, const float* obj_pos,
                          const float* obj_quat, const int32_t* geom_type, const float* geom_params, float* depth, void* stream) {
  // sizes first: nothing below this block runs, and no CUDA call is made, for a request the static scratch cannot hold
  if (n_envs <= 0 || n_links <= 0 || n_taxels <= 0) return fail(nullptr, TS_ERR_INVALID_ARG, "ts_depth_static: sizes must be positive");
  if ((long long)n_envs * n_links > (long long)TS_STATIC_MAX_FRAMES)
    return fail(nullptr, TS_ERR_INVALID_ARG, "ts_depth_static: n_envs * n_links = " + std::to_string((long long)n_envs * n_links) +
                " exceeds TS_STATIC_MAX_FRAMES = " + std::to_string((long long)TS_STATIC_MAX_FRAMES) +
                " (the static scratch array holds " + std::to_string((long long)TS_STATIC_SCRATCH_BYTES) + " bytes)");
  if ((long long)n_envs * n_taxels >= (1LL << 40)) return fail(nullptr, TS_ERR_INVALID_ARG, "ts_depth_static: n_envs * n_taxels too large");
  if (!taxel_pos || !taxel_radius || !taxel_link || !link_pos || !link_quat || !obj_pos || !obj_quat || !geom_type || !geom_params || !depth)
    return fail(nullptr, TS_ERR_INVALID_ARG, "ts_depth_static: null pointer");
  if ((reinterpret_cast<uintptr_t>(geom_params) & 15u) || (reinterpret_cast<uintptr_t>(link_quat) & 15u) || (reinterpret_cast<uintptr_t>(obj_quat) & 15u))
    return fail(nullptr, TS_ERR_INVALID_ARG, "ts_depth_static: link_quat, obj_quat and geom_params must be 16-byte aligned");
  const cudaError_t e = (cudaError_t)ts_static_depth_launch(n_envs, n_links, n_taxels, taxel_pos, taxel_radius, taxel_link, link_pos, link_quat,
                                                            obj_pos, obj_quat, geom_type, geom_params, depth, stream);
  if (e != cudaSuccess) return cuda_fail(nullptr, e, "ts_depth_static");
  return TS_OK;
}

// ---- checkpoint / resume ----------------------------------------------------------------------------------------
namespace {
constexpr int kStateSections = 15;
struct StateHeader {            // 160 bytes
  uint64_t magic, total;
  uint32_t version, n_envs, n_taxels, tp, nh, n_markers, ring_slots, pc_n, n_patches, objs, gstep, n_sections;
  uint64_t section_bytes[kStateSections];
};
static_assert(sizeof(StateHeader) == 16 + 48 + 8 * kStateSections, "StateHeader layout");
constexpr uint64_t kStateMagic = 0x3130455441545354ull;  // "TSSTATE01"
struct StateSection { void* dev; uint64_t bytes; };

// Every array a ctx carries across steps, in blob order.  Absent ones (feature off) have 0 bytes.
void state_sections(const ts_ctx* c, StateSection s[kStateSections], uint32_t* ring_slots) {
  const uint64_t E = (uint64_t)c->cfg.n_envs, T = (uint64_t)c->T, M = (uint64_t)c->M, Tp = (uint64_t)c->Tp;
  const uint32_t S = c->st_ring ? (uint32_t)(c->cfg.read_delay + c->cfg.read_jitter) : 0u;
  const uint64_t nsh = c->sh_on ? E * (uint64_t)c->P * (uint64_t)c->cfg.objs_per_env * (uint64_t)((c->pc_n + 15) / 16 * 16) : 0;
  *ring_slots = S;
  s[0] = {c->st_flags, E * T};
  s[1] = {c->reset_step, sizeof(uint32_t) * E};
  s[2] = {c->episode, sizeof(uint32_t) * E};
  s[3] = {c->st_hyst, c->st_hyst ? sizeof(float) * E * (uint64_t)c->nh * Tp : 0};
  s[4] = {c->st_drift, c->st_drift ? sizeof(float) * E * 6 * Tp : 0};
  s[5] = {c->st_ring, sizeof(float) * E * 6 * Tp * S};
  s[6] = {c->sn_h, c->sn_h ? sizeof(float4) * E * T : 0};
  s[7] = {c->sn_d, c->sn_d ? sizeof(float2) * E * T : 0};
  s[8] = {c->sm_h, c->sm_h ? sizeof(float) * E * M * 6 : 0};
  s[9] = {c->sm_d, c->sm_d ? sizeof(float) * E * M * 3 : 0};
  s[10] = {c->sh_on, nsh};
  s[11] = {c->sh_e, sizeof(float4) * nsh};
  const uint64_t Sr = (uint64_t)(c->cfg.read_delay + c->cfg.read_jitter);
  s[12] = {c->sn_ring, c->sn_ring ? sizeof(float2) * E * Sr * T : 0};
  s[13] = {c->sm_ring, c->sm_ring ? sizeof(float) * E * Sr * M * 3 : 0};
  s[14] = {c->sh_cnt, c->sh_cnt ? sizeof(int32_t) * E * (uint64_t)c->P * (uint64_t)c->cfg.objs_per_env : 0};
}

StateHeader state_header(const ts_ctx* c, const StateSection s[kStateSections], uint32_t ring_slots) {
  StateHeader h = {};
  h.magic = kStateMagic; h.version = 1;
  h.n_envs = (uint32_t)c->cfg.n_envs; h.n_taxels = (uint32_t)c->T; h.tp = (uint32_t)c->Tp; h.nh = (uint32_t)c->nh;
  h.n_markers = (uint32_t)c->M; h.ring_slots = ring_slots; h.pc_n = c->sh_on ? (uint32_t)c->pc_n : 0u;
  h.n_patches = (uint32_t)c->P; h.objs = (uint32_t)c->cfg.objs_per_env; h.gstep = c->gstep; h.n_sections = kStateSections;
  h.total = sizeof(StateHeader);
  for (int i = 0; i < kStateSections; ++i) { h.section_bytes[i] = s[i].bytes; h.total += (s[i].bytes + 15) & ~(uint64_t)15; }
  return h;
}
}  // namespace

ts_status ts_state_bytes(const ts_ctx* c, uint64_t* bytes) {
  if (!c || !bytes) return TS_ERR_INVALID_ARG;
  StateSection s[kStateSections]; uint32_t S;
  state_sections(c, s, &S);
  *bytes = state_header(c, s, S).total;
  return TS_OK;
}

ts_status ts_get_state(ts_ctx* c, void* host_buf, uint64_t capacity, void* stream) {
  if (!c) return TS_ERR_INVALID_ARG;
  if (!host_buf) return fail(c, TS_ERR_INVALID_ARG, "ts_get_state: null buffer");
  DeviceGuard guard(c->device);
  StateSection s[kStateSections]; uint32_t S;
  state_sections(c, s, &S);
  const StateHeader h = state_header(c, s, S);
  if (capacity < h.total) return fail(c, TS_ERR_INVALID_ARG, "ts_get_state: buffer smaller than ts_state_bytes");
  std::memcpy(host_buf, &h, sizeof(h));
  uint64_t off = sizeof(h);
  for (int i = 0; i < kStateSections; ++i) {
    if (s[i].bytes) TS_CUDA(c, cudaMemcpyAsync((char*)host_buf + off, s[i].dev, s[i].bytes, cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    off += (s[i].bytes + 15) & ~(uint64_t)15;
  }
  TS_CUDA(c, cudaStreamSynchronize((cudaStream_t)stream));
  return TS_OK;
}

ts_status ts_set_state(ts_ctx* c, const void* host_buf, uint64_t bytes, void* stream) {
  if (!c) return TS_ERR_INVALID_ARG;
  if (!host_buf || bytes < sizeof(StateHeader)) return fail(c, TS_ERR_INVALID_ARG, "ts_set_state: no header");
  DeviceGuard guard(c->device);
  StateSection s[kStateSections]; uint32_t S;
  state_sections(c, s, &S);
  const StateHeader want = state_header(c, s, S);
  StateHeader h;
  std::memcpy(&h, host_buf, sizeof(h));
  if (h.magic != kStateMagic || h.version != 1) return fail(c, TS_ERR_INVALID_ARG, "ts_set_state: not a ts state blob");
  bool same = h.total == want.total && bytes >= h.total && h.n_envs == want.n_envs && h.n_taxels == want.n_taxels && h.tp == want.tp &&
              h.nh == want.nh && h.n_markers == want.n_markers && h.ring_slots == want.ring_slots && h.pc_n == want.pc_n &&
              h.n_patches == want.n_patches && h.objs == want.objs && h.n_sections == want.n_sections;
  for (int i = 0; same && i < kStateSections; ++i) same = h.section_bytes[i] == want.section_bytes[i];
  if (!same) return fail(c, TS_ERR_INVALID_ARG, "ts_set_state: blob was taken from a ctx with another configuration");
  uint64_t off = sizeof(h);
  for (int i = 0; i < kStateSections; ++i) {
    if (s[i].bytes) TS_CUDA(c, cudaMemcpyAsync(s[i].dev, (const char*)host_buf + off, s[i].bytes, cudaMemcpyHostToDevice, (cudaStream_t)stream));
    off += (s[i].bytes + 15) & ~(uint64_t)15;
  }
  TS_CUDA(c, cudaStreamSynchronize((cudaStream_t)stream));
  c->gstep = h.gstep;
  return TS_OK;
}

ts_status ts_kernel_times_ms(ts_ctx* c, float* out_ms, int32_t capacity, int32_t* n_steps) {
  if (!c) return TS_ERR_INVALID_ARG;
  DeviceGuard guard(c->device);
  const int n = (int)(c->ev_used / 4);
  for (int i = 0; i < n && i < capacity && out_ms; ++i) {
    cudaEvent_t* ev = &c->ev[(size_t)4 * i];
    TS_CUDA(c, cudaEventSynchronize(ev[3]));
    if (c->timing_detail) {
      for (int k = 0; k < 3; ++k) TS_CUDA(c, cudaEventElapsedTime(out_ms + 4 * i + k, ev[k], ev[k + 1]));
    } else {  // enable = 1: one pair of events around the whole step (reported in the step-kernel column)
      out_ms[4 * i] = 0.f; out_ms[4 * i + 2] = 0.f;
      TS_CUDA(c, cudaEventElapsedTime(out_ms + 4 * i + 1, ev[0], ev[3]));
    }
    unsigned long long ck[2] = {0, 0};
    TS_CUDA(c, cudaMemcpy(ck, c->clock_buf + 2 * i, sizeof(ck), cudaMemcpyDeviceToHost));
    out_ms[4 * i + 3] = ck[1] > ck[0] ? (float)((double)(ck[1] - ck[0]) * 1e-6) : 0.f;
  }
  if (n_steps) *n_steps = n;
  return TS_OK;
}

ts_status ts_kernel_time_ms(ts_ctx* c, int32_t enable, float* mean_ms, int32_t* n_steps) {
  if (!c) return TS_ERR_INVALID_ARG;
  DeviceGuard guard(c->device);
  double sum = 0.0, sum1 = 0.0;
  const int n = (int)(c->ev_used / 4);
  for (int i = 0; i < n; ++i) {
    cudaEvent_t* ev = &c->ev[(size_t)4 * i];
    TS_CUDA(c, cudaEventSynchronize(ev[3]));
    float ms = 0.f, ms1 = 0.f;
    TS_CUDA(c, cudaEventElapsedTime(&ms, ev[0], ev[3]));
    if (c->timing_detail) TS_CUDA(c, cudaEventElapsedTime(&ms1, ev[0], ev[2]));
    else ms1 = ms;
    sum += ms; sum1 += ms1;
  }
  c->last_first_kernel_ms = n ? (float)(sum1 / n) : 0.f;
  c->ev_used = 0;
  if (enable) {                    // device-side clock slots: {first block start (min), last block end (max)}
    if (!c->clock_buf) TS_CUDA(c, cudaMalloc((void**)&c->clock_buf, sizeof(unsigned long long) * 2 * TS_TIMING_MAX_STEPS));
    std::vector<unsigned long long> init((size_t)2 * TS_TIMING_MAX_STEPS);
    for (int i = 0; i < TS_TIMING_MAX_STEPS; ++i) { init[2 * i] = ~0ULL; init[2 * i + 1] = 0ULL; }
    TS_CUDA(c, cudaMemcpy(c->clock_buf, init.data(), sizeof(unsigned long long) * init.size(), cudaMemcpyHostToDevice));
  }
  if (enable && c->ev.empty()) {   // the pool is created here, never inside ts_step
    c->ev.reserve((size_t)4 * TS_TIMING_MAX_STEPS);
    for (int i = 0; i < 4 * TS_TIMING_MAX_STEPS; ++i) {
      cudaEvent_t a;
      TS_CUDA(c, cudaEventCreate(&a));
      c->ev.push_back(a);
    }
  }
  c->timing = enable != 0;
  c->timing_detail = enable == 2;
  if (mean_ms) *mean_ms = n ? (float)(sum / n) : 0.f;
  if (n_steps) *n_steps = n;
  return TS_OK;
}

float ts_first_kernel_time_ms(const ts_ctx* c) { return c ? c->last_first_kernel_ms : 0.f; }

ts_status ts_destroy(ts_ctx* c) {
  if (!c) return TS_OK;
  {
    DeviceGuard guard(c->device);
    cudaDeviceSynchronize();
    free_all(c);
  }
  delete c;
  return TS_OK;
}

}  // extern "C"
