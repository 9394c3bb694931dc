// ORACLE -- TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, obviously-correct CPU implementation of the batched tactile readout of
// Tactile Genesis (arxiv/paper_2606_22332), written from /root/reference/PAPER.md
// ("P:NNN" = PAPER.md line NNN) and the readings fixed in DESIGN.md / SURVEY.md 8(c)
// ("O0".."O8", "D1".."D5", "Q1".."Q24").  Every floating-point step is evaluated in
// double precision on the fp32 input values, in the paper's order and notation; there
// is no blocking, fusion, table or reordering.  It shares no code with the CUDA path
// (paper_2606_22332_b200/csrc/), includes none of its headers and is never imported by
// the product.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may load it.
//
// Pins (tests/test_oracle_pins.py, all -m "not gpu"):
//   philox4x32_10            known-answer vectors (P15)
//   primitive SDFs           closed forms + brute-force surface sampling (P1, P5)
//   grid SDF                 affine field exact, star grid vs analytic, brute-force mesh (P6, P7, P9)
//   depth / contact          worked sphere example, Schmitt hand sequence (P1, P10)
//   kinematic force/torque   closed-form spring / damping / cap values (P2-P4)
//   marker                   single-source closed form at r* (P11)
//   march                    plane closed form t_k = D/cos(th) (1-(1-cos th)^k) (P12)
//   noise                    Maxwell / asym closed forms, crosstalk patch-sum, drift moments, dead (P13-P16)
//   remaining A.8 knobs      bias / white-noise moments, quantisation levels and hand values, per-episode gain,
//                            stuck readout range and constancy (P19-P22; readings R1-R4 in DESIGN.md)
//   radius noise (Eq. 26)    eps = d~ - d read back from |f| = k_n d^alpha: range, moments, the Philox word,
//                            reach limits, constancy per episode, the max(0, .) clamp (P24; reading R8)
//   read delay (Eq. 25)      delayed run = undelayed run shifted by Delta steps, zeros while the pipe fills and
//                            after a reset; additive terms not delayed; jitter value unique per (env, step), all
//                            values reached, one draw reproduced from the Philox word (P25; reading R9)
//   whole path               rigid-frame invariance, filler slots, no-contact zeros (P8, P17)
// parity unpinned: none of the functions; the *joint* output on star grids with all
// stages on (configs 4-5) is pinned only through the per-stage pins above (P18).
//
// Build: g++ -O2 -std=c++17 -fPIC -shared -fopenmp oracle.cpp -o liboracle.so

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <deque>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

struct V3 { double x, y, z; };
inline V3 operator+(V3 a, V3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
inline V3 operator-(V3 a, V3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
inline V3 operator*(double s, V3 a) { return {s * a.x, s * a.y, s * a.z}; }
inline double dot(V3 a, V3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
inline V3 cross(V3 a, V3 b) { return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }
inline double norm(V3 a) { return std::sqrt(dot(a, a)); }
inline V3 ld3(const float* p) { return {(double)p[0], (double)p[1], (double)p[2]}; }

// O0: rotation matrix of a quaternion (w,x,y,z), used as given (no renormalisation).
struct M3 { double m[3][3]; };
inline M3 quat_to_R(const float* q) {
  double w = q[0], x = q[1], y = q[2], z = q[3];
  M3 R;
  R.m[0][0] = 1 - 2 * (y * y + z * z); R.m[0][1] = 2 * (x * y - w * z);     R.m[0][2] = 2 * (x * z + w * y);
  R.m[1][0] = 2 * (x * y + w * z);     R.m[1][1] = 1 - 2 * (x * x + z * z); R.m[1][2] = 2 * (y * z - w * x);
  R.m[2][0] = 2 * (x * z - w * y);     R.m[2][1] = 2 * (y * z + w * x);     R.m[2][2] = 1 - 2 * (x * x + y * y);
  return R;
}
inline V3 mul(const M3& R, V3 v) {
  return {R.m[0][0] * v.x + R.m[0][1] * v.y + R.m[0][2] * v.z,
          R.m[1][0] * v.x + R.m[1][1] * v.y + R.m[1][2] * v.z,
          R.m[2][0] * v.x + R.m[2][1] * v.y + R.m[2][2] * v.z};
}
inline V3 mulT(const M3& R, V3 v) {  // R^T v
  return {R.m[0][0] * v.x + R.m[1][0] * v.y + R.m[2][0] * v.z,
          R.m[0][1] * v.x + R.m[1][1] * v.y + R.m[2][1] * v.z,
          R.m[0][2] * v.x + R.m[1][2] * v.y + R.m[2][2] * v.z};
}

// ---------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al. 2011).  O8 "Random draws".
// ---------------------------------------------------------------------------------
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// O8: u = (2 (w >> 9) + 1) 2^-24, in (0,1), exact in fp32.
inline double word_to_uniform(uint32_t w) { return (2.0 * (double)(w >> 9) + 1.0) * (1.0 / 16777216.0); }

// O8: Box-Muller on a word pair.
inline void box_muller(uint32_t wa, uint32_t wb, double* z0, double* z1) {
  const double two_pi = 6.283185307179586476925286766559;
  double ua = word_to_uniform(wa), ub = word_to_uniform(wb);
  double r = std::sqrt(-2.0 * std::log(ua));
  *z0 = r * std::cos(two_pi * ub);
  *z1 = r * std::sin(two_pi * ub);
}

// ---------------------------------------------------------------------------------
// O2: geometry queries.  Types: 0 none, 1 sphere, 2 box, 3 capsule, 4 SDF grid.
// ---------------------------------------------------------------------------------
enum { G_NONE = 0, G_SPHERE = 1, G_BOX = 2, G_CAPSULE = 3, G_GRID = 4 };

struct Query {
  double phi;      // signed distance
  V3 g;            // object-frame gradient, NOT normalised
  double face;     // grid only: min over axes of the distance (voxels) of u to an integer
  double boxgap;   // box interior only: gap between the two largest w_i
};

// sphere: phi = |x| - r, g = x/|x|  (Q7: g = e_z at the centre)
Query sdf_sphere(V3 x, double r) {
  Query q; q.face = INFINITY; q.boxgap = INFINITY;
  double n = norm(x);
  q.phi = n - r;
  q.g = (n < 1e-12) ? V3{0, 0, 1} : (1.0 / n) * x;
  return q;
}

// box, half-extents b (Q7)
Query sdf_box(V3 x, V3 b) {
  Query q; q.face = INFINITY; q.boxgap = INFINITY;
  double w[3] = {std::fabs(x.x) - b.x, std::fabs(x.y) - b.y, std::fabs(x.z) - b.z};
  double sgn[3] = {x.x < 0 ? -1.0 : 1.0, x.y < 0 ? -1.0 : 1.0, x.z < 0 ? -1.0 : 1.0};
  double p[3] = {std::fmax(w[0], 0.0), std::fmax(w[1], 0.0), std::fmax(w[2], 0.0)};
  double lp = std::sqrt(p[0] * p[0] + p[1] * p[1] + p[2] * p[2]);
  double wmax = std::fmax(w[0], std::fmax(w[1], w[2]));
  q.phi = lp + std::fmin(wmax, 0.0);
  bool outside = (w[0] > 0) || (w[1] > 0) || (w[2] > 0);
  if (outside) {
    q.g = {sgn[0] * p[0] / lp, sgn[1] * p[1] / lp, sgn[2] * p[2] / lp};
  } else {
    int i = 0;                       // argmax w_i, ties -> lowest index
    if (w[1] > w[i]) i = 1;
    if (w[2] > w[i]) i = 2;
    double second = -INFINITY;
    for (int a = 0; a < 3; ++a) if (a != i) second = std::fmax(second, w[a]);
    q.boxgap = w[i] - second;
    q.g = {0, 0, 0};
    if (i == 0) q.g.x = sgn[0]; else if (i == 1) q.g.y = sgn[1]; else q.g.z = sgn[2];
  }
  return q;
}

// capsule, radius r, half-length h along local z
Query sdf_capsule(V3 x, double r, double h) {
  Query q; q.face = INFINITY; q.boxgap = INFINITY;
  double zc = std::fmin(std::fmax(x.z, -h), h);
  V3 y = {x.x, x.y, x.z - zc};
  double n = norm(y);
  q.phi = n - r;
  q.g = (n < 1e-12) ? V3{0, 0, 1} : (1.0 / n) * y;
  return q;
}

// grid: N^3 nodes, voxel hv, node i at origin + i hv with origin = -(N-1)/2 hv; data
// index (k N + j) N + i, i <-> x fastest.  Trilinear value, exact gradient of the
// interpolant in cell i0, outside-grid extension phi = phi_tri(u_c) + |x - x(u_c)|.
Query sdf_grid(V3 x, const float* data, int N, double hv) {
  Query q; q.boxgap = INFINITY;
  double origin = -0.5 * (N - 1) * hv;
  double xs[3] = {x.x, x.y, x.z};
  double uc[3], f[3];
  int i0[3];
  double face = INFINITY, out2 = 0.0;
  for (int a = 0; a < 3; ++a) {
    double u = (xs[a] - origin) / hv;
    double c = std::fmin(std::fmax(u, 0.0), (double)(N - 1));
    uc[a] = c;
    int i = (int)std::floor(c);
    if (i > N - 2) i = N - 2;
    i0[a] = i;
    f[a] = c - i;
    double xc = origin + c * hv;
    out2 += (xs[a] - xc) * (xs[a] - xc);
    face = std::fmin(face, std::fabs(u - std::round(u)));
  }
  auto at = [&](int di, int dj, int dk) -> double {
    size_t idx = ((size_t)(i0[2] + dk) * N + (size_t)(i0[1] + dj)) * N + (size_t)(i0[0] + di);
    return (double)data[idx];
  };
  double c000 = at(0, 0, 0), c100 = at(1, 0, 0), c010 = at(0, 1, 0), c110 = at(1, 1, 0);
  double c001 = at(0, 0, 1), c101 = at(1, 0, 1), c011 = at(0, 1, 1), c111 = at(1, 1, 1);
  double fx = f[0], fy = f[1], fz = f[2];
  double gx0 = 1 - fx, gy0 = 1 - fy, gz0 = 1 - fz;
  double tri = c000 * gx0 * gy0 * gz0 + c100 * fx * gy0 * gz0 + c010 * gx0 * fy * gz0 + c110 * fx * fy * gz0 +
               c001 * gx0 * gy0 * fz + c101 * fx * gy0 * fz + c011 * gx0 * fy * fz + c111 * fx * fy * fz;
  double dx = ((c100 - c000) * gy0 * gz0 + (c110 - c010) * fy * gz0 + (c101 - c001) * gy0 * fz + (c111 - c011) * fy * fz) / hv;
  double dy = ((c010 - c000) * gx0 * gz0 + (c110 - c100) * fx * gz0 + (c011 - c001) * gx0 * fz + (c111 - c101) * fx * fz) / hv;
  double dz = ((c001 - c000) * gx0 * gy0 + (c101 - c100) * fx * gy0 + (c011 - c010) * gx0 * fy + (c111 - c110) * fx * fy) / hv;
  q.phi = tri + std::sqrt(out2);
  q.g = {dx, dy, dz};
  q.face = face;
  return q;
}

// Closest point of triangle (a, b, c) to p: the Voronoi-region walk of Ericson, "Real-Time Collision Detection" 5.1.5,
// restated (vertex regions, edge regions, face).
V3 closest_point_triangle(V3 p, V3 a, V3 b, V3 c) {
  V3 ab = b - a, ac = c - a, ap = p - a;
  double d1 = dot(ab, ap), d2 = dot(ac, ap);
  if (d1 <= 0.0 && d2 <= 0.0) return a;
  V3 bp = p - b;
  double d3 = dot(ab, bp), d4 = dot(ac, bp);
  if (d3 >= 0.0 && d4 <= d3) return b;
  double vc = d1 * d4 - d3 * d2;
  if (vc <= 0.0 && d1 >= 0.0 && d3 <= 0.0) return a + (d1 / (d1 - d3)) * ab;
  V3 cp = p - c;
  double d5 = dot(ab, cp), d6 = dot(ac, cp);
  if (d6 >= 0.0 && d5 <= d6) return c;
  double vb = d5 * d2 - d1 * d6;
  if (vb <= 0.0 && d2 >= 0.0 && d6 <= 0.0) return a + (d2 / (d2 - d6)) * ac;
  double va = d3 * d6 - d5 * d4;
  if (va <= 0.0 && (d4 - d3) >= 0.0 && (d5 - d6) >= 0.0) return b + ((d4 - d3) / ((d4 - d3) + (d5 - d6))) * (c - b);
  double denom = 1.0 / (va + vb + vc);
  return a + (vb * denom) * ab + (vc * denom) * ac;
}

// Ray (orig, unit dir) against triangle (a, b, c), both faces (Moeller-Trumbore, restated): hit distance t >= 0, or -1.
double ray_triangle(V3 orig, V3 dir, V3 a, V3 b, V3 c) {
  V3 e1 = b - a, e2 = c - a, pv = cross(dir, e2);
  double det = dot(e1, pv);
  if (std::fabs(det) < 1e-300) return -1.0;
  double inv = 1.0 / det;
  V3 tv = orig - a;
  double u = dot(tv, pv) * inv;
  if (u < 0.0 || u > 1.0) return -1.0;
  V3 qv = cross(tv, e1);
  double v = dot(dir, qv) * inv;
  if (v < 0.0 || u + v > 1.0) return -1.0;
  double t = dot(e2, qv) * inv;
  return t >= 0.0 ? t : -1.0;
}

struct Geom {
  int type;
  double p[4];
  const float* grid;  // type 4
  int N;
  double hv;
};

Query sdf_eval(const Geom& g, V3 x) {
  switch (g.type) {
    case G_SPHERE: return sdf_sphere(x, g.p[0]);
    case G_BOX: return sdf_box(x, {g.p[0], g.p[1], g.p[2]});
    case G_CAPSULE: return sdf_capsule(x, g.p[0], g.p[1]);
    case G_GRID: return sdf_grid(x, g.grid, g.N, g.hv);
    default: {
      Query q; q.phi = INFINITY; q.g = {0, 0, 1}; q.face = INFINITY; q.boxgap = INFINITY;
      return q;
    }
  }
}

// ---------------------------------------------------------------------------------
// Parameters and patches (plain C structs, mirrored by ctypes in oracle/oracle.py)
// ---------------------------------------------------------------------------------
extern "C" {
typedef struct orc_patch {
  int32_t link;
  float origin[3];
  float u_axis[3];
  float v_axis[3];
  float size_u, size_v;
  int32_t nu, nv;
  float radius;
  int32_t marker_nu, marker_nv;
} orc_patch;

typedef struct orc_params {
  float k_n, c_n, alpha, k_t, k_omega, mu, eta_on, eta_off;
  int32_t use_velocity;
  float s_d, lambda_d, alpha_e, c_e;
  float r_prox;
  int32_t march_steps;
  float dt;
  int32_t noise_enable;
  uint32_t seed_lo, seed_hi;
  float sigma_rw_force, sigma_rw_torque;
  int32_t hyst_mode;  // 0 off, 1 Maxwell (Eq. 29-30), 2 asymmetric first-order (D3)
  float beta, tau, alpha_load, alpha_unload;
  float p_dead, chi;
  // remaining knobs of App. A.8 (readings R1-R4)
  float sigma_white_force, sigma_white_torque;  // Eq. 25 n_t ~ N(0, sigma^2), channels 0-2 / 3-5
  float bias_force, bias_torque;                // Eq. 25 constant bias b
  float quant_force, quant_torque;              // Eq. 25 quantisation step q (0 = off)
  float gain_min, gain_max;                     // Eq. 27 per-reset gain gamma_bj ~ U[min, max] (1, 1 = off)
  float stuck_min_force, stuck_max_force, stuck_min_torque, stuck_max_torque;  // Eq. 28 stuck readout z_bj ~ U[l, u]
  float xtalk_sigma;  // Eq. 11 / 31: 0 = 4-neighbour stencil (D4); > 0 = Gaussian G_sigma, sigma in taxel pitches (R7)
  float radius_noise; // Eq. 26: rho (metres), R~_j = max(0, R_j + eps_j), eps_j ~ U[-rho, rho] (R8); 0 = off
  int32_t read_delay, read_jitter;  // Eq. 25 Delta_read in steps and its uniform jitter +-J steps (R9); 0, 0 = off
  // Noisy readouts of the scalar sensors (Table 3: ContactDepth, Proximity, Elastomer take every knob but
  // crosstalk; values Table 12; reading R10): per class {depth, prox, marker}
  // white sigma, random-walk sigma, bias, quantisation step, stuck range [l, u]
  float sn_sigma_white[3], sn_sigma_rw[3], sn_bias[3], sn_quant[3], sn_stuck_min[3], sn_stuck_max[3];
  // Point-cloud ProximityTaxel (App. A.6, Eq. 12-17): sensing radius R_j, k, k_s, density scalar
  // (0.01 m, 300, 10, 100)
  float pc_radius, pc_k, pc_ks, pc_density;
  // Elastomer shear history (App. A.7, Eq. 22-23; constants P:304: s_s = 100, lambda_s = 2000,
  // eta_enter = 1e-5 m, eta_exit = 1e-4 m); shear_enable adds sum_p u^s_pj to the marker output (reading R11)
  int32_t shear_enable;
  float s_s, lambda_s, eta_enter, eta_exit;
} orc_params;
}

struct Oracle {
  int E, L, K, T, P, M;
  std::vector<int64_t> env_id;  // global env ids (Philox counters use these)
  orc_params prm;
  // S0 layout; values are the fp32-rounded ones, held in double.
  std::vector<V3> pos, nrm, mpos, mnrm;
  std::vector<double> radius;
  std::vector<int> link, patch, iu, iv, mpatch;
  std::vector<int> p_start, p_nu, p_nv, p_link, p_mstart, p_mcount;
  std::vector<double> p_eps;
  std::vector<int> nbr;  // [T,4]: -u, +u, -v, +v; -1 = none
  // geometry
  std::vector<Geom> geom;  // [E,K]
  std::vector<float> bank;
  int bank_n = 0, bank_N = 0;
  double bank_hv = 0;
  // state
  std::vector<uint8_t> ybit;                // Schmitt state [E,T]
  std::vector<double> hyst_a, hyst_b, drift;  // [E,T,6]: (xi, x_prev) or (y, -)
  double* aux_quant = nullptr;                // [E,T,6] comparator aid, see orc_set_aux_quant
  double* aux_rgate = nullptr;                // [E,T] comparator aid, see orc_set_aux_rgate
  double* aux_wingap = nullptr;               // [E,T] comparator aid, see orc_set_aux_wingap
  // noisy scalar readouts (R10): outputs and comparator aids handed in by orc_set_scalar_noisy; state
  double *depth_noisy = nullptr, *prox_noisy = nullptr, *marker_noisy = nullptr;   // [E,T], [E,T], [E,M,3]
  double *aux_sq_depth = nullptr, *aux_sq_prox = nullptr, *aux_sq_marker = nullptr, *aux_sasym_marker = nullptr;
  std::vector<double> sn_ha, sn_hb, sn_dr;    // [E,T,2] depth, prox: hysteresis (xi | y), x_prev, drift
  std::vector<double> sm_ha, sm_hb, sm_dr;    // [E,M,3] marker channels
  // point-cloud ProximityTaxel (A.6): bank of surface point clouds in the object frame, cloud id per (env, object)
  std::vector<float> pc_pts;                  // [G,N,3]
  int pc_G = 0, pc_N = 0;
  std::vector<int32_t> pc_id;                 // [E,K], -1 = the object is not tracked
  double* proxpc = nullptr;                   // [E,T,6] output handed in by orc_set_proxpc
  // elastomer shear history (Eq. 22): anchor per (env, patch, object, tracked point), link frame
  std::vector<uint8_t> sh_on;                 // [E,P,K,N] anchored?
  std::vector<V3> sh_e;                       // [E,P,K,N] anchor e_p
  std::vector<V3> p_center, p_ua, p_va;       // [P] pad centre and unit axes (fp32 values), link frame
  std::vector<double> p_su, p_sv;             // [P] pad extents
  // raycast depth backend (App. A.1): bank of triangle meshes in the object frame, mesh of each (env, object)
  std::vector<float> rc_verts;                // all vertices [sum V, 3]
  std::vector<int32_t> rc_tris;               // all triangles [sum F, 3], vertex indices local to their mesh
  std::vector<int32_t> rc_voff, rc_toff;      // [G + 1] offsets
  std::vector<int32_t> rc_id;                 // [E,K], -1 = no mesh
  double *rc_depth = nullptr, *rc_nrm = nullptr, *rc_gap = nullptr;   // [E,T], [E,T,3], [E,T] outputs handed in by orc_set_raycast_out
  std::vector<std::deque<std::vector<double>>> hist;  // [E] the last Delta + J post-crosstalk fields [T,6] of the episode
  std::vector<std::deque<std::vector<double>>> shist;  // [E] the same for the scalar readouts (R10): post-hysteresis depth [T], prox [T], markers [M,3]
  std::vector<uint32_t> n_step, episode;      // [E]
};

inline double f32(double v) { return (double)(float)v; }

// S0 (Q19): cell-centred regular grid on each patch.
void build_layout(Oracle& o, const orc_patch* patches, int P, int T, const uint8_t* link_mask) {
  o.P = P; o.T = T;
  o.pos.assign(T, {0, 0, 0}); o.nrm.assign(T, {0, 0, 1}); o.radius.assign(T, 0.0);
  o.link.assign(T, 0); o.patch.assign(T, -1); o.iu.assign(T, 0); o.iv.assign(T, 0);
  o.nbr.assign((size_t)T * 4, -1);
  o.mpos.clear(); o.mnrm.clear(); o.mpatch.clear();
  o.p_center.clear(); o.p_ua.clear(); o.p_va.clear(); o.p_su.clear(); o.p_sv.clear();
  o.p_start.clear(); o.p_nu.clear(); o.p_nv.clear(); o.p_link.clear(); o.p_mstart.clear(); o.p_mcount.clear(); o.p_eps.clear();
  int t = 0;
  for (int p = 0; p < P; ++p) {
    const orc_patch& d = patches[p];
    V3 org = ld3(d.origin), ua = ld3(d.u_axis), va = ld3(d.v_axis);
    V3 n = cross(ua, va);
    bool keep = (link_mask == nullptr) || link_mask[d.link];
    o.p_start.push_back(t); o.p_nu.push_back(d.nu); o.p_nv.push_back(d.nv); o.p_link.push_back(d.link);
    o.p_eps.push_back(f32((double)d.size_u / d.nu));
    o.p_center.push_back(org); o.p_ua.push_back(ua); o.p_va.push_back(va);
    o.p_su.push_back((double)d.size_u); o.p_sv.push_back((double)d.size_v);
    for (int v = 0; v < d.nv; ++v)
      for (int u = 0; u < d.nu; ++u, ++t) {
        double su = ((u + 0.5) / d.nu - 0.5) * (double)d.size_u;
        double sv = ((v + 0.5) / d.nv - 0.5) * (double)d.size_v;
        V3 x = org + su * ua + sv * va;
        o.pos[t] = {f32(x.x), f32(x.y), f32(x.z)};
        o.nrm[t] = {f32(n.x), f32(n.y), f32(n.z)};
        o.radius[t] = keep ? (double)d.radius : 0.0;   // link filter -> filler
        o.link[t] = d.link; o.patch[t] = p; o.iu[t] = u; o.iv[t] = v;
        o.nbr[(size_t)t * 4 + 0] = (u > 0) ? t - 1 : -1;
        o.nbr[(size_t)t * 4 + 1] = (u < d.nu - 1) ? t + 1 : -1;
        o.nbr[(size_t)t * 4 + 2] = (v > 0) ? t - d.nu : -1;
        o.nbr[(size_t)t * 4 + 3] = (v < d.nv - 1) ? t + d.nu : -1;
      }
    o.p_mstart.push_back((int)o.mpos.size());
    o.p_mcount.push_back(d.marker_nu * d.marker_nv);
    for (int v = 0; v < d.marker_nv; ++v)
      for (int u = 0; u < d.marker_nu; ++u) {
        double su = ((u + 0.5) / d.marker_nu - 0.5) * (double)d.size_u;
        double sv = ((v + 0.5) / d.marker_nv - 0.5) * (double)d.size_v;
        V3 x = org + su * ua + sv * va;
        o.mpos.push_back({f32(x.x), f32(x.y), f32(x.z)});
        o.mnrm.push_back({f32(n.x), f32(n.y), f32(n.z)});
        o.mpatch.push_back(p);
      }
  }
  o.M = (int)o.mpos.size();
  // slots t..T-1 stay fillers with R = 0 (Q18)
}

// O5 (Eq. 4-10, D2, Q4-Q6): kinematic force / torque of one taxel, link frame.
void kinematic_ft(const orc_params& pr, double d, V3 m_world, V3 q, V3 x_j, const M3& RL, V3 pL, V3 vL, V3 wL,
                  V3 pO, V3 vO, V3 wO, double out[6]) {
  for (int c = 0; c < 6; ++c) out[c] = 0.0;
  if (!(d > 0.0)) return;                                    // Q5: every term gated on d > 0
  V3 mbar = mulT(RL, m_world);                               // m_bar = R_L^T m
  double s = std::pow(d, (double)pr.alpha);                  // s_j = d^alpha
  V3 f, tau;
  if (pr.use_velocity) {
    V3 vC = vO + cross(wO, q - pO);                          // Eq. 4, r_C = p_O (Q4)
    V3 vLq = vL + cross(wL, q - pL);                         // Eq. 5, r_L = p_L
    V3 vrel = mulT(RL, vC - vLq);                            // Eq. 6
    double vn_s = dot(vrel, mbar);
    V3 vn = vn_s * mbar;                                     // Eq. 7
    V3 vt = vrel - vn;
    V3 fn = ((double)pr.k_n * s) * mbar + ((double)pr.c_n * s) * vn;  // Eq. 8 normal part
    V3 ft = (-(double)pr.k_t) * vt;                          // Eq. 8 tangential part
    double lim = (double)pr.mu * norm(fn);                   // D2: Coulomb cap (mu = inf -> Eq. 8)
    double nft = norm(ft);
    if (nft > lim) ft = (lim / nft) * ft;
    f = fn + ft;
    tau = cross(x_j, f) - ((double)pr.k_omega * dot(wO - wL, m_world)) * mbar;   // Eq. 9
  } else {
    f = ((double)pr.k_n * s) * mbar;
    tau = cross(x_j, f);
  }
  out[0] = f.x; out[1] = f.y; out[2] = f.z; out[3] = tau.x; out[4] = tau.y; out[5] = tau.z;
}

// O7 (D1): bounded march along a from q through phi = min_k phi_k.
template <class PhiFn>
double march(PhiFn phi, double r_prox, int steps) {
  double t = 0.0;
  for (int i = 0; i < steps; ++i) {
    double s = phi(t);
    t = std::fmin(t + std::fmax(s, 0.0), r_prox);
  }
  return r_prox - t;
}

}  // namespace

// =================================================================================
// C interface (ctypes)
// =================================================================================
extern "C" {

void orc_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }

double orc_uniform(uint32_t w) { return word_to_uniform(w); }

void orc_box_muller(uint32_t wa, uint32_t wb, double* z) { box_muller(wa, wb, &z[0], &z[1]); }

// One geometry query in the object frame: out = {phi, gx, gy, gz (unnormalised), face, boxgap}.
void orc_sdf_query(int type, const double* params, const float* grid, int N, double hv, const double* x, double* out) {
  Geom g; g.type = type; for (int i = 0; i < 4; ++i) g.p[i] = params ? params[i] : 0.0;
  g.grid = grid; g.N = N; g.hv = hv;
  Query q = sdf_eval(g, {x[0], x[1], x[2]});
  out[0] = q.phi; out[1] = q.g.x; out[2] = q.g.y; out[3] = q.g.z; out[4] = q.face; out[5] = q.boxgap;
}

void* orc_create(const orc_params* prm, const orc_patch* patches, int n_patches, int n_taxels, const uint8_t* link_mask,
                 int n_envs, const int64_t* env_ids, int n_links, int objs_per_env) {
  int need = 0;
  for (int p = 0; p < n_patches; ++p) need += patches[p].nu * patches[p].nv;
  if (need > n_taxels || n_envs <= 0) return nullptr;
  Oracle* o = new Oracle();
  o->prm = *prm;
  o->E = n_envs; o->L = n_links; o->K = objs_per_env;
  o->env_id.resize(n_envs);
  for (int e = 0; e < n_envs; ++e) o->env_id[e] = env_ids ? env_ids[e] : e;
  build_layout(*o, patches, n_patches, n_taxels, link_mask);
  size_t ET = (size_t)o->E * o->T;
  o->ybit.assign(ET, 0);
  o->hyst_a.assign(ET * 6, 0.0); o->hyst_b.assign(ET * 6, 0.0); o->drift.assign(ET * 6, 0.0);   // Q12
  o->n_step.assign(o->E, 0); o->episode.assign(o->E, 0);
  o->hist.assign(o->E, {});
  o->shist.assign(o->E, {});
  o->sn_ha.assign(ET * 2, 0.0); o->sn_hb.assign(ET * 2, 0.0); o->sn_dr.assign(ET * 2, 0.0);
  { size_t EM = (size_t)o->E * o->M * 3; o->sm_ha.assign(EM, 0.0); o->sm_hb.assign(EM, 0.0); o->sm_dr.assign(EM, 0.0); }
  Geom none; none.type = G_NONE; none.grid = nullptr; none.N = 0; none.hv = 0; for (double& v : none.p) v = 0;
  o->geom.assign((size_t)o->E * o->K, none);
  return o;
}

void orc_destroy(void* h) { delete (Oracle*)h; }

int orc_n_markers(void* h) { return ((Oracle*)h)->M; }

// Copies the S0 layout out for inspection (any pointer may be NULL).
void orc_get_layout(void* h, double* pos, double* nrm, double* radius, int32_t* link, int32_t* patch, int32_t* nbr,
                    double* mpos, double* mnrm, int32_t* mpatch) {
  Oracle& o = *(Oracle*)h;
  for (int t = 0; t < o.T; ++t) {
    if (pos) { pos[3 * t] = o.pos[t].x; pos[3 * t + 1] = o.pos[t].y; pos[3 * t + 2] = o.pos[t].z; }
    if (nrm) { nrm[3 * t] = o.nrm[t].x; nrm[3 * t + 1] = o.nrm[t].y; nrm[3 * t + 2] = o.nrm[t].z; }
    if (radius) radius[t] = o.radius[t];
    if (link) link[t] = o.link[t];
    if (patch) patch[t] = o.patch[t];
    if (nbr) for (int a = 0; a < 4; ++a) nbr[4 * t + a] = o.nbr[(size_t)4 * t + a];
  }
  for (int j = 0; j < o.M; ++j) {
    if (mpos) { mpos[3 * j] = o.mpos[j].x; mpos[3 * j + 1] = o.mpos[j].y; mpos[3 * j + 2] = o.mpos[j].z; }
    if (mnrm) { mnrm[3 * j] = o.mnrm[j].x; mnrm[3 * j + 1] = o.mnrm[j].y; mnrm[3 * j + 2] = o.mnrm[j].z; }
    if (mpatch) mpatch[j] = o.mpatch[j];
  }
}

// Geometry: type[E,K], params[E,K,4] (sphere r; box hx,hy,hz; capsule r,h; grid id in params[0]),
// bank[n_grids,N,N,N] fp32 x-fastest (copied).
int orc_set_geometry(void* h, const int32_t* type, const float* params, int n_grids, int N, float voxel, const float* bank) {
  Oracle& o = *(Oracle*)h;
  o.bank_n = n_grids; o.bank_N = N; o.bank_hv = (double)voxel;
  size_t per = (size_t)N * N * N;
  o.bank.assign(bank, bank + per * (size_t)n_grids);
  for (size_t i = 0; i < (size_t)o.E * o.K; ++i) {
    Geom g; g.type = type[i]; g.grid = nullptr; g.N = N; g.hv = (double)voxel;
    for (int a = 0; a < 4; ++a) g.p[a] = (double)params[4 * i + a];
    if (g.type == G_GRID) {
      int id = (int)params[4 * i];
      if (id < 0 || id >= n_grids) return 1;
      g.grid = o.bank.data() + per * (size_t)id;
    }
    o.geom[i] = g;
  }
  return 0;
}

// ts_reset semantics (8b): zero the state of the masked envs, restart their step count,
// advance their episode (which re-draws the dead mask).
void orc_reset(void* h, const uint8_t* env_mask) {
  Oracle& o = *(Oracle*)h;
  for (int e = 0; e < o.E; ++e) {
    if (env_mask && !env_mask[e]) continue;
    for (int t = 0; t < o.T; ++t) {
      size_t i = (size_t)e * o.T + t;
      o.ybit[i] = 0;
      for (int c = 0; c < 6; ++c) { o.hyst_a[i * 6 + c] = 0; o.hyst_b[i * 6 + c] = 0; o.drift[i * 6 + c] = 0; }
    }
    o.n_step[e] = 0;
    o.episode[e] += 1;
    o.hist[e].clear();
    o.shist[e].clear();
    if (!o.sh_on.empty()) {
      size_t per = (size_t)o.P * o.K * o.pc_N;
      std::fill(o.sh_on.begin() + (size_t)e * per, o.sh_on.begin() + (size_t)(e + 1) * per, (uint8_t)0);
    }
    for (size_t i = (size_t)e * o.T * 2; i < (size_t)(e + 1) * o.T * 2; ++i) { o.sn_ha[i] = 0; o.sn_hb[i] = 0; o.sn_dr[i] = 0; }
    for (size_t i = (size_t)e * o.M * 3; i < (size_t)(e + 1) * o.M * 3; ++i) { o.sm_ha[i] = 0; o.sm_hb[i] = 0; o.sm_dr[i] = 0; }
  }
}

// O8 dead mask (Eq. 28, D5): stream 2, n = 0, word0 < floor(p_dead 2^32).
static bool is_dead(const Oracle& o, int e, int t) {
  if (!o.prm.noise_enable) return false;
  uint32_t thr = (uint32_t)std::floor((double)o.prm.p_dead * 4294967296.0);
  uint32_t ctr[4] = {(uint32_t)o.env_id[e], (uint32_t)t, 0u, (o.episode[e] << 4) | 2u};
  uint32_t key[2] = {o.prm.seed_lo, o.prm.seed_hi};
  uint32_t w[4];
  philox4x32_10(ctr, key, w);
  return w[0] < thr;
}

// R10: one channel of a noisy scalar readout (Eq. 25, 27-30; no crosstalk, Table 3):
//   x = gamma * clean -> hysteresis (Eq. 29-30 or ASYM) -> y = h + b + sigma_w z_w + D, D <- D + sigma_rw z_rw
//   -> quantize(y, q) -> a dead probe reads its stuck value.  Returns the readout; aq / aa receive the comparator aids
// (distance to the nearest rounding boundary; |x| - |y_prev| where the signs differ), +inf where not applicable.
static double scalar_chain(const orc_params& pr, int cls, double clean, double gain, bool is_dead, double stuck_u,
                           double z_rw, double z_w, double& ha, double& hb, double& drift, double decay,
                           double* aq, double* aa, const double* delayed = nullptr, double* hrec = nullptr) {
  double x = gain * clean, hval = x;
  if (aa) *aa = INFINITY;
  if (pr.hyst_mode == 1) {                                        // Eq. 29-30
    double xi = decay * ha + (x - hb);
    ha = xi; hb = x;
    hval = x + (double)pr.beta * xi;
  } else if (pr.hyst_mode == 2) {                                 // D3, Q14
    double yp = ha;
    if (aa && x * yp < 0.0) *aa = std::fabs(x) - std::fabs(yp);
    double al = (std::fabs(x) > std::fabs(yp)) ? (double)pr.alpha_load : (double)pr.alpha_unload;
    double y = yp + al * (x - yp);
    ha = y;
    hval = y;
  }
  // Eq. 25 read delay (R9 / R10): only the signal is delayed, y_{t - Delta_n}; bias, white noise and drift are those
  // of step t.  hrec receives this step's signal for the history, delayed points at the one to show (NULL: Delta_n = 0).
  if (hrec) *hrec = hval;
  if (delayed) hval = *delayed;
  drift += (double)pr.sn_sigma_rw[cls] * z_rw;                    // Eq. 25 d_t = d_{t-1} + w_t
  double y = hval + (double)pr.sn_bias[cls] + (double)pr.sn_sigma_white[cls] * z_w + drift;
  if (aq) *aq = INFINITY;
  float q = pr.sn_quant[cls];
  if (q > 0.0f) {                                                 // quantize(., q) as R5: decision in fp32
    float yf = (float)y, r = yf / q, k = std::nearbyintf(r);
    if (aq) *aq = (0.5 - std::fabs((double)r - (double)k)) * (double)q;
    y = (double)(k * q);
  }
  if (is_dead) y = (double)pr.sn_stuck_min[cls] + ((double)pr.sn_stuck_max[cls] - (double)pr.sn_stuck_min[cls]) * stuck_u;
  return y;
}

// One step of the whole path.  Inputs fp32 [E,L,*] / [E,K,*]; outputs double (NULL = skip).
// aux (all optional): aux_phi[E,T] = min_k phi_k(q_j); aux_face[E,T] = voxel-face distance of the
// winner if it is a grid (else +inf); aux_boxgap[E,T]; aux_asym[E,T,6] = |x|-|y_prev| where the
// signs of x and y_prev differ (else +inf) -- used only for the comparator's band accounting.
void orc_step(void* h, const float* link_pos, const float* link_quat, const float* link_linvel, const float* link_angvel,
              const float* obj_pos, const float* obj_quat, const float* obj_linvel, const float* obj_angvel,
              uint8_t* contact, double* depth, double* ft, double* marker, double* prox, double* ft_noisy, uint8_t* dead,
              double* aux_phi, double* aux_face, double* aux_boxgap, double* aux_asym, int n_threads) {
  Oracle& o = *(Oracle*)h;
  const orc_params& pr = o.prm;
  const int T = o.T, L = o.L, K = o.K, M = o.M;
  (void)n_threads;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(n_threads > 0 ? n_threads : 1)
#endif
  for (int e = 0; e < o.E; ++e) {
    std::vector<double> phi_min(T), dep(T), ftc((size_t)T * 6), ftn((size_t)T * 6), hcl((size_t)T * 6);
    std::vector<double> dep_t(T, 0.0), prox_c(T, 0.0), marker_c((size_t)M * 3, 0.0);   // inputs of the noisy scalar readouts (R10)
    std::vector<uint8_t> deadv(T, 0);
    for (int j = 0; j < T; ++j) {
      size_t ej = (size_t)e * T + j;
      bool active = o.radius[j] > 0.0;                       // R_j = 0 -> filler
      int l = o.link[j];
      const float* lp = link_pos + ((size_t)e * L + l) * 3;
      M3 RL = quat_to_R(link_quat + ((size_t)e * L + l) * 4);
      V3 pL = ld3(lp);
      V3 q = pL + mul(RL, o.pos[j]);                         // Eq. 1
      V3 a = mul(RL, o.nrm[j]);
      // O2/O3: query all K objects, winner = max_k [R - phi_k]_+, ties -> lowest k
      double best_phi = INFINITY; int kstar = -1; Query qstar{}; M3 RO_star{};
      double second_phi = INFINITY;                          // comparator aid only (winner ties when K > 1)
      for (int k = 0; k < K; ++k) {
        const Geom& g = o.geom[(size_t)e * K + k];
        if (g.type == G_NONE) continue;
        V3 pO = ld3(obj_pos + ((size_t)e * K + k) * 3);
        M3 RO = quat_to_R(obj_quat + ((size_t)e * K + k) * 4);
        V3 xo = mulT(RO, q - pO);
        Query r = sdf_eval(g, xo);
        if (r.phi < best_phi) { second_phi = best_phi; best_phi = r.phi; kstar = k; qstar = r; RO_star = RO; }
        else if (r.phi < second_phi) second_phi = r.phi;
      }
      phi_min[j] = best_phi;
      if (o.aux_wingap) o.aux_wingap[ej] = second_phi - best_phi;   // +inf with fewer than two objects
      double d = (active && kstar >= 0) ? std::fmax(0.0, o.radius[j] - best_phi) : 0.0;   // Eq. 2
      dep[j] = d;
      dep_t[j] = d;
      if (aux_phi) aux_phi[ej] = best_phi;
      if (aux_face) aux_face[ej] = kstar >= 0 ? qstar.face : INFINITY;
      if (aux_boxgap) aux_boxgap[ej] = kstar >= 0 ? qstar.boxgap : INFINITY;
      // O4 (Eq. 3): Schmitt trigger, strict >
      uint8_t y = 0;
      if (active) y = (d > (double)pr.eta_on) || (o.ybit[ej] == 1 && d > (double)pr.eta_off);
      o.ybit[ej] = y;
      deadv[j] = active && is_dead(o, e, j);
      if (contact) contact[ej] = deadv[j] ? 0 : y;
      if (dead) dead[ej] = deadv[j];
      if (depth) depth[ej] = d;
      // O5
      double f6[6] = {0, 0, 0, 0, 0, 0};
      if (active && d > 0.0) {
        double gn = norm(qstar.g);
        V3 m = (gn < 1e-12) ? (-1.0) * a : (1.0 / gn) * mul(RO_star, qstar.g);   // Q2
        V3 pO = ld3(obj_pos + ((size_t)e * K + kstar) * 3);
        kinematic_ft(pr, d, m, q, o.pos[j], RL, pL, ld3(link_linvel + ((size_t)e * L + l) * 3),
                     ld3(link_angvel + ((size_t)e * L + l) * 3), pO, ld3(obj_linvel + ((size_t)e * K + kstar) * 3),
                     ld3(obj_angvel + ((size_t)e * K + kstar) * 3), f6);
      }
      for (int c = 0; c < 6; ++c) { ftc[(size_t)j * 6 + c] = f6[c]; if (ft) ft[ej * 6 + c] = f6[c]; }
      // Eq. 26 (R8): the NOISY readout senses with the perturbed radius R~_j = max(0, R_j + eps_j),
      // eps_j ~ U[-rho, rho] drawn once per (env, taxel, episode): stream 8, n = 0, word 0.  The clean
      // outputs above keep R_j; the noise chain below starts from the Eq. 4-9 readout at depth
      // d~ = [R~_j - phi]_+ (same winner, same contact normal).
      double g6[6] = {f6[0], f6[1], f6[2], f6[3], f6[4], f6[5]};
      if (o.aux_rgate) o.aux_rgate[ej] = INFINITY;
      if (pr.noise_enable && pr.radius_noise != 0.0f && active) {
        uint32_t key[2] = {pr.seed_lo, pr.seed_hi}, w[4];
        uint32_t cr[4] = {(uint32_t)o.env_id[e], (uint32_t)j, 0u, (o.episode[e] << 4) | 8u};
        philox4x32_10(cr, key, w);
        double rho = (double)pr.radius_noise;
        double eps = -rho + 2.0 * rho * word_to_uniform(w[0]);
        double Rt = std::fmax(0.0, o.radius[j] + eps);
        double dt_ = (kstar >= 0) ? std::fmax(0.0, Rt - best_phi) : 0.0;
        if (o.aux_rgate) o.aux_rgate[ej] = std::fabs(Rt - best_phi);
        dep_t[j] = dt_;                                          // the noisy depth readout senses with R~_j too
        for (int c = 0; c < 6; ++c) g6[c] = 0.0;
        if (dt_ > 0.0) {
          double gn = norm(qstar.g);
          V3 m = (gn < 1e-12) ? (-1.0) * a : (1.0 / gn) * mul(RO_star, qstar.g);   // Q2
          V3 pO = ld3(obj_pos + ((size_t)e * K + kstar) * 3);
          kinematic_ft(pr, dt_, m, q, o.pos[j], RL, pL, ld3(link_linvel + ((size_t)e * L + l) * 3),
                       ld3(link_angvel + ((size_t)e * L + l) * 3), pO, ld3(obj_linvel + ((size_t)e * K + kstar) * 3),
                       ld3(obj_angvel + ((size_t)e * K + kstar) * 3), g6);
        }
      }
      for (int c = 0; c < 6; ++c) ftn[(size_t)j * 6 + c] = g6[c];
      // O7
      if (prox) {
        double P = 0.0;
        if (active) {
          auto phi_at = [&](double t) {
            double best = INFINITY;
            V3 x = q + t * a;
            for (int k = 0; k < K; ++k) {
              const Geom& g = o.geom[(size_t)e * K + k];
              if (g.type == G_NONE) continue;
              V3 pO = ld3(obj_pos + ((size_t)e * K + k) * 3);
              M3 RO = quat_to_R(obj_quat + ((size_t)e * K + k) * 4);
              best = std::fmin(best, sdf_eval(g, mulT(RO, x - pO)).phi);
            }
            return best;
          };
          P = march(phi_at, (double)pr.r_prox, pr.march_steps);
        }
        prox[ej] = P;
        prox_c[j] = P;
      }
      // A.6 point-cloud ProximityTaxel.  Tracked points p_i = p_O + R_O p_i^o of every tracked object;
      // P_j = {i : |p_i - q_j| < R_j} (Eq. 12 set), P_ij = R_j - |p_i - q_j| (Eq. 12), point / taxel velocities with
      // r_i = p_O, r_L = p_L (Eq. 13, Q4), tangential part (Eq. 14), density scale rho_b = density / max(N_active_b, 1)
      // with N_active_b = tracked points of env b (Eq. 15, reading Q27), world force / torque (Eq. 16-17), reported
      // as R_L^T f^w, R_L^T tau^w.
      if (o.proxpc) {
        double out6[6] = {0, 0, 0, 0, 0, 0};
        if (active && o.pc_N > 0) {
          long n_active = 0;
          for (int k = 0; k < K; ++k) if (o.pc_id[(size_t)e * K + k] >= 0) n_active += o.pc_N;
          const double rho = (double)pr.pc_density / (double)std::max(n_active, 1L);
          const double Rj = (double)pr.pc_radius;
          V3 vL = ld3(link_linvel + ((size_t)e * L + l) * 3), wL = ld3(link_angvel + ((size_t)e * L + l) * 3);
          V3 vtax = vL + cross(wL, q - pL);                                  // Eq. 13
          V3 fw = {0, 0, 0}, tw = {0, 0, 0};
          for (int k = 0; k < K; ++k) {
            const int id = o.pc_id[(size_t)e * K + k];
            if (id < 0) continue;
            V3 pO = ld3(obj_pos + ((size_t)e * K + k) * 3);
            M3 RO = quat_to_R(obj_quat + ((size_t)e * K + k) * 4);
            V3 vO = ld3(obj_linvel + ((size_t)e * K + k) * 3), wO = ld3(obj_angvel + ((size_t)e * K + k) * 3);
            const float* pts = o.pc_pts.data() + (size_t)id * o.pc_N * 3;
            for (int i = 0; i < o.pc_N; ++i) {
              V3 pi = pO + mul(RO, ld3(pts + 3 * i));
              V3 dv = pi - q;
              double dist = norm(dv);
              if (!(dist < Rj)) continue;                                    // P_j
              double P = Rj - dist;                                          // Eq. 12
              V3 vp = vO + cross(wO, pi - pO);                               // Eq. 13
              V3 vr = vp - vtax;
              V3 vt = vr - dot(vr, a) * a;                                   // Eq. 14
              fw = fw + ((double)pr.pc_k * rho * P) * a + ((double)pr.pc_ks * rho * P) * vt;   // Eq. 16
              tw = tw + ((double)pr.pc_k * rho * P) * cross(dv, a);          // Eq. 17
            }
          }
          V3 fl = mulT(RL, fw), tl = mulT(RL, tw);
          out6[0] = fl.x; out6[1] = fl.y; out6[2] = fl.z; out6[3] = tl.x; out6[4] = tl.y; out6[5] = tl.z;
        }
        for (int c = 0; c < 6; ++c) o.proxpc[ej * 6 + c] = out6[c];
      }
      // A.1 raycast depth backend, brute force over every triangle of every meshed object (the BVH of the
      // paper only prunes candidates): sphere-triangle closest-point test, penetration = R_j - dist, and ray-triangle
      // test from q_j along -a_j, penetration = R_j - hit_distance (reading Q28: ray from the probe centre, both
      // faces); the deepest of all wins, the normal is the winning triangle's face normal (object winding), reported in
      // the sensor-link frame.  rc_gap = margin to the best triangle with a DIFFERENT normal (comparator aid).
      if (o.rc_depth) {
        double best = 0.0, second = 0.0;
        V3 bn = {0, 0, 0};
        if (active) {
          const double Rj = o.radius[j];
          for (int k = 0; k < K; ++k) {
            const int id = o.rc_id.empty() ? -1 : o.rc_id[(size_t)e * K + k];
            if (id < 0) continue;
            V3 pO = ld3(obj_pos + ((size_t)e * K + k) * 3);
            M3 RO = quat_to_R(obj_quat + ((size_t)e * K + k) * 4);
            V3 qo = mulT(RO, q - pO), ao = mulT(RO, a);
            const float* V = o.rc_verts.data() + (size_t)o.rc_voff[id] * 3;
            for (int f = o.rc_toff[id]; f < o.rc_toff[id + 1]; ++f) {
              V3 A = ld3(V + 3 * o.rc_tris[3 * f]), B = ld3(V + 3 * o.rc_tris[3 * f + 1]), C3 = ld3(V + 3 * o.rc_tris[3 * f + 2]);
              double pen = 0.0;
              double dist = norm(qo - closest_point_triangle(qo, A, B, C3));
              if (dist < Rj) pen = Rj - dist;
              double th = ray_triangle(qo, (-1.0) * ao, A, B, C3);
              if (th >= 0.0 && th < Rj) pen = std::fmax(pen, Rj - th);
              if (!(pen > 0.0)) continue;
              V3 fn = cross(B - A, C3 - A);
              double fl = norm(fn);
              V3 nw = fl > 0.0 ? mulT(RL, mul(RO, (1.0 / fl) * fn)) : V3{0, 0, 0};   // link frame
              if (pen > best) {
                if (norm(nw - bn) > 1e-6) second = best;
                best = pen; bn = nw;
              } else if (pen > second && norm(nw - bn) > 1e-6) {
                second = pen;
              }
            }
          }
        }
        o.rc_depth[ej] = best;
        if (o.rc_nrm) { o.rc_nrm[ej * 3] = bn.x; o.rc_nrm[ej * 3 + 1] = bn.y; o.rc_nrm[ej * 3 + 2] = bn.z; }
        if (o.rc_gap) o.rc_gap[ej] = best - second;
      }
    }
    // O6 (Eq. 18-21, 23 first sum; Q15-Q17): dilation of each patch's markers by its active taxels
    if (marker) {
      double lam = (double)pr.lambda_d, cE = (double)pr.c_e;
      double gbar = std::exp(-0.5) / std::sqrt(2.0 * lam);
      for (int jm = 0; jm < M; ++jm) {
        int p = o.mpatch[jm];
        double eps = o.p_eps[p], rhobar = 1.0 / (2.0 * eps);
        V3 u = {0, 0, 0};
        V3 nj = o.mnrm[jm];
        int n = o.p_nu[p] * o.p_nv[p];
        for (int i = o.p_start[p]; i < o.p_start[p] + n; ++i) {
          if (!(o.radius[i] > 0.0)) continue;
          double hi = std::fmax(0.0, -phi_min[i]);                       // Eq. 19
          V3 z = o.mpos[jm] - o.pos[i];
          V3 r = z - dot(z, nj) * nj;                                   // Eq. 18
          double r2 = dot(r, r);
          double g = std::exp(-lam * r2);
          double rho = 1.0 / (r2 + eps * eps);
          double w = hi * (cE * g / gbar + (1.0 - cE) * rho / rhobar);   // Eq. 20
          double bulge = (hi > 0.0) ? std::pow(hi, (double)pr.alpha_e) * g : 0.0;
          u = u + (double)pr.s_d * (w * r + bulge * nj);                 // Eq. 21
        }
        size_t o3 = ((size_t)e * M + jm) * 3;
        marker[o3] = u.x; marker[o3 + 1] = u.y; marker[o3 + 2] = u.z;
        marker_c[(size_t)jm * 3] = u.x; marker_c[(size_t)jm * 3 + 1] = u.y; marker_c[(size_t)jm * 3 + 2] = u.z;
      }
      // Eq. 22-23 (R11): anchored shear history of the tracked surface points.  For every patch (elastomer pad) and
      // tracked point p: z_p = R_L^T (p_O + R_O p^o - p_L) (sensor-link frame); elastomer SDF of a flat pad
      // phi_el = n . (z_p - x_c) over the pad (|u| <= size_u / 2, |v| <= size_v / 2), +inf beside it; the anchor
      // e_p = z_p is set when phi_el < -eta_enter and cleared when phi_el > +eta_exit; h_p = max(0, -phi_el);
      // u^s_pj = s_s Pi_n(z_p - e_p) h_p exp(-lambda_s |Pi_n(x_j - z_p)|^2) is added to every marker j of the patch.
      if (pr.shear_enable && o.pc_N > 0) {
        const int P = o.P, N = o.pc_N;
        for (int pi = 0; pi < P; ++pi) {
          if (o.p_mcount[pi] == 0 || !(o.radius[o.p_start[pi]] > 0.0)) continue;     // no markers / filtered-out link
          const int l = o.p_link[pi];
          M3 RL = quat_to_R(link_quat + ((size_t)e * L + l) * 4);
          V3 pL = ld3(link_pos + ((size_t)e * L + l) * 3);
          V3 n = o.mnrm[o.p_mstart[pi]];
          for (int k = 0; k < K; ++k) {
            const int id = o.pc_id[(size_t)e * K + k];
            if (id < 0) continue;
            V3 pO = ld3(obj_pos + ((size_t)e * K + k) * 3);
            M3 RO = quat_to_R(obj_quat + ((size_t)e * K + k) * 4);
            const float* pts = o.pc_pts.data() + (size_t)id * N * 3;
            for (int i = 0; i < N; ++i) {
              size_t si = (((size_t)e * P + pi) * K + k) * N + i;
              V3 z = mulT(RL, pO + mul(RO, ld3(pts + 3 * i)) - pL);
              V3 rel = z - o.p_center[pi];
              double phi_el = INFINITY;
              if (std::fabs(dot(rel, o.p_ua[pi])) <= 0.5 * o.p_su[pi] && std::fabs(dot(rel, o.p_va[pi])) <= 0.5 * o.p_sv[pi])
                phi_el = dot(rel, n);
              if (!o.sh_on[si] && phi_el < -(double)pr.eta_enter) { o.sh_on[si] = 1; o.sh_e[si] = z; }
              else if (o.sh_on[si] && phi_el > (double)pr.eta_exit) o.sh_on[si] = 0;
              if (!o.sh_on[si]) continue;
              double hp = std::fmax(0.0, -phi_el);
              if (!(hp > 0.0)) continue;
              V3 dz = z - o.sh_e[si];
              V3 dzt = dz - dot(dz, n) * n;                                           // Pi_n(z_p - e_p)
              for (int jm = o.p_mstart[pi]; jm < o.p_mstart[pi] + o.p_mcount[pi]; ++jm) {
                V3 r = o.mpos[jm] - z;
                V3 rt = r - dot(r, n) * n;                                            // Pi_n(x_j - z_p)
                double wgt = (double)pr.s_s * hp * std::exp(-(double)pr.lambda_s * dot(rt, rt));   // Eq. 22
                size_t o3 = ((size_t)e * M + jm) * 3;
                marker[o3] += wgt * dzt.x; marker[o3 + 1] += wgt * dzt.y; marker[o3 + 2] += wgt * dzt.z;   // Eq. 23
                marker_c[(size_t)jm * 3] += wgt * dzt.x; marker_c[(size_t)jm * 3 + 1] += wgt * dzt.y; marker_c[(size_t)jm * 3 + 2] += wgt * dzt.z;
              }
            }
          }
        }
      }
    }
    // O8: hysteresis -> crosstalk -> drift -> dead
    if (pr.noise_enable) {
      uint32_t n = o.n_step[e];
      double decay = std::exp(-(double)pr.dt / (double)pr.tau);
      // Eq. 25 read delay (R9): the readout at step n shows the post-crosstalk signal of step n - Delta_n,
      // Delta_n = max(0, Delta + k_n), k_n uniform on {-J..J}, one draw per (env, step) shared by all taxels:
      // stream 9, taxel counter 0xffffffff, k_n = (((word0 >> 9) * (2J + 1)) >> 23) - J.  Steps before the
      // episode began read 0 (Q12).
      const bool delay_on = pr.read_delay > 0 || pr.read_jitter > 0;
      int delta_n = 0;
      std::vector<double> cfield;
      if (delay_on) {
        int k_n = 0;
        if (pr.read_jitter > 0) {
          uint32_t key[2] = {pr.seed_lo, pr.seed_hi}, w[4];
          uint32_t cj[4] = {(uint32_t)o.env_id[e], 0xffffffffu, n, (o.episode[e] << 4) | 9u};
          philox4x32_10(cj, key, w);
          k_n = (int)(((uint64_t)(w[0] >> 9) * (uint64_t)(2 * pr.read_jitter + 1)) >> 23) - pr.read_jitter;
        }
        delta_n = std::max(0, pr.read_delay + k_n);
        cfield.assign((size_t)T * 6, 0.0);
      }
      for (int j = 0; j < T; ++j) {
        size_t ej = (size_t)e * T + j;
        // Eq. 27 (R2): per-unit calibration gain, drawn once per (env, taxel, episode): stream 3, n = 0, word 0
        double gain = 1.0;
        if (o.radius[j] > 0.0 && (pr.gain_min != 1.0f || pr.gain_max != 1.0f)) {
          uint32_t key[2] = {pr.seed_lo, pr.seed_hi}, w[4];
          uint32_t cg[4] = {(uint32_t)o.env_id[e], (uint32_t)j, 0u, (o.episode[e] << 4) | 3u};
          philox4x32_10(cg, key, w);
          gain = (double)pr.gain_min + ((double)pr.gain_max - (double)pr.gain_min) * word_to_uniform(w[0]);
        }
        for (int c = 0; c < 6; ++c) {
          double x = gain * ftn[(size_t)j * 6 + c], hval = x;
          if (aux_asym) aux_asym[ej * 6 + c] = INFINITY;
          if (o.radius[j] > 0.0) {
            if (pr.hyst_mode == 1) {                                      // Eq. 29-30
              double xi = decay * o.hyst_a[ej * 6 + c] + (x - o.hyst_b[ej * 6 + c]);
              o.hyst_a[ej * 6 + c] = xi; o.hyst_b[ej * 6 + c] = x;
              hval = x + (double)pr.beta * xi;
            } else if (pr.hyst_mode == 2) {                               // D3, Q14
              double yp = o.hyst_a[ej * 6 + c];
              if (aux_asym && x * yp < 0.0) aux_asym[ej * 6 + c] = std::fabs(x) - std::fabs(yp);
              double al = (std::fabs(x) > std::fabs(yp)) ? (double)pr.alpha_load : (double)pr.alpha_unload;
              double y = yp + al * (x - yp);
              o.hyst_a[ej * 6 + c] = y;
              hval = y;
            }
          }
          hcl[(size_t)j * 6 + c] = hval;
        }
      }
      for (int j = 0; j < T; ++j) {
        size_t ej = (size_t)e * T + j;
        bool active = o.radius[j] > 0.0;
        // draws: stream 0 -> channels 0-3, stream 1 words 0-1 -> channels 4-5
        double z[6] = {0, 0, 0, 0, 0, 0};
        if (active) {
          uint32_t key[2] = {pr.seed_lo, pr.seed_hi}, w0[4], w1[4];
          uint32_t c0[4] = {(uint32_t)o.env_id[e], (uint32_t)j, n, (o.episode[e] << 4) | 0u};
          uint32_t c1[4] = {(uint32_t)o.env_id[e], (uint32_t)j, n, (o.episode[e] << 4) | 1u};
          philox4x32_10(c0, key, w0);
          philox4x32_10(c1, key, w1);
          box_muller(w0[0], w0[1], &z[0], &z[1]);
          box_muller(w0[2], w0[3], &z[2], &z[3]);
          box_muller(w1[0], w1[1], &z[4], &z[5]);
        }
        // Eq. 25 white noise n_t (R3): streams 6 / 7 of the same counter, laid out like the drift draws
        double zw[6] = {0, 0, 0, 0, 0, 0};
        if (active && (pr.sigma_white_force != 0.0f || pr.sigma_white_torque != 0.0f)) {
          uint32_t key[2] = {pr.seed_lo, pr.seed_hi}, w0[4], w1[4];
          uint32_t c0[4] = {(uint32_t)o.env_id[e], (uint32_t)j, n, (o.episode[e] << 4) | 6u};
          uint32_t c1[4] = {(uint32_t)o.env_id[e], (uint32_t)j, n, (o.episode[e] << 4) | 7u};
          philox4x32_10(c0, key, w0);
          philox4x32_10(c1, key, w1);
          box_muller(w0[0], w0[1], &zw[0], &zw[1]);
          box_muller(w0[2], w0[3], &zw[2], &zw[3]);
          box_muller(w1[0], w1[1], &zw[4], &zw[5]);
        }
        // Eq. 28 stuck readout z_bj (R4): streams 4 / 5, n = 0; only dead taxels use it
        double stuck[6] = {0, 0, 0, 0, 0, 0};
        if (active && deadv[j]) {
          uint32_t key[2] = {pr.seed_lo, pr.seed_hi}, w0[4], w1[4];
          uint32_t c0[4] = {(uint32_t)o.env_id[e], (uint32_t)j, 0u, (o.episode[e] << 4) | 4u};
          uint32_t c1[4] = {(uint32_t)o.env_id[e], (uint32_t)j, 0u, (o.episode[e] << 4) | 5u};
          philox4x32_10(c0, key, w0);
          philox4x32_10(c1, key, w1);
          const uint32_t ww[6] = {w0[0], w0[1], w0[2], w0[3], w1[0], w1[1]};
          for (int c = 0; c < 6; ++c) {
            double lo = c < 3 ? (double)pr.stuck_min_force : (double)pr.stuck_min_torque;
            double hi = c < 3 ? (double)pr.stuck_max_force : (double)pr.stuck_max_torque;
            stuck[c] = lo + (hi - lo) * word_to_uniform(ww[c]);
          }
        }
        for (int c = 0; c < 6; ++c) {
          double out = 0.0;
          if (o.aux_quant) o.aux_quant[ej * 6 + c] = INFINITY;
          if (active) {
            double hj = hcl[(size_t)j * 6 + c];
            double cj;
            if (pr.xtalk_sigma > 0.0f) {
              // Eq. 11 / 31 (R7): z~ = (1 - chi) z + chi (G_sigma * z) on the patch grid.  G_sigma[du, dv] =
              // g[du] g[dv], g[d] = exp(-d^2 / (2 sigma^2)) for |d| <= r = ceil(3 sigma), L1-normalised over
              // its full support; plain convolution, zero outside the patch (inactive sources count as 0).
              const double sg = (double)pr.xtalk_sigma;
              const int r = (int)std::ceil(3.0 * sg);
              double norm = 0.0;
              for (int d = -r; d <= r; ++d) norm += std::exp(-(double)(d * d) / (2.0 * sg * sg));
              const int pj = o.patch[j], nu = o.p_nu[pj], nv = o.p_nv[pj], u0 = o.iu[j], v0 = o.iv[j];
              double conv = 0.0;
              for (int dv = -r; dv <= r; ++dv)
                for (int du = -r; du <= r; ++du) {
                  const int u = u0 + du, v = v0 + dv;
                  if (u < 0 || u >= nu || v < 0 || v >= nv) continue;
                  const int k = o.p_start[pj] + v * nu + u;
                  if (!(o.radius[k] > 0.0)) continue;
                  const double w = std::exp(-(double)(du * du) / (2.0 * sg * sg)) / norm *
                                   (std::exp(-(double)(dv * dv) / (2.0 * sg * sg)) / norm);
                  conv += w * hcl[(size_t)k * 6 + c];
                }
              cj = (1.0 - (double)pr.chi) * hj + (double)pr.chi * conv;
            } else {
              double acc = 0.0;                                           // D4, Q11
              for (int a = 0; a < 4; ++a) {
                int k = o.nbr[(size_t)j * 4 + a];
                if (k >= 0 && o.radius[k] > 0.0) acc += hcl[(size_t)k * 6 + c] - hj;
              }
              cj = hj + ((double)pr.chi / 4.0) * acc;
            }
            if (delay_on) {                                               // Eq. 25 y_{t - Delta_read} (R9)
              cfield[(size_t)j * 6 + c] = cj;
              const int have = (int)o.hist[e].size();                     // earlier steps of this episode still held
              if (delta_n > 0) cj = (delta_n <= have) ? o.hist[e][have - delta_n][(size_t)j * 6 + c] : 0.0;
            }
            double sig = (c < 3) ? (double)pr.sigma_rw_force : (double)pr.sigma_rw_torque;
            double D = o.drift[ej * 6 + c] + sig * z[c];                  // Eq. 25 drift
            o.drift[ej * 6 + c] = D;
            double sw = (c < 3) ? (double)pr.sigma_white_force : (double)pr.sigma_white_torque;
            double bias = (c < 3) ? (double)pr.bias_force : (double)pr.bias_torque;
            double y = cj + bias + sw * zw[c] + D;                        // Eq. 25 before quantisation (R1)
            float q = (c < 3) ? pr.quant_force : pr.quant_torque;
            if (q > 0.0f) {
              // Eq. 25 quantize(., q): the integer decision is taken in fp32 (the precision of the readout):
              // k = rint(y / q) on the fp32 image of y, round half to even; result k q in fp32.
              float yf = (float)y;
              float r = yf / q;
              float k = std::nearbyintf(r);
              if (o.aux_quant) o.aux_quant[ej * 6 + c] = (0.5 - std::fabs((double)r - (double)k)) * (double)q;
              y = (double)(k * q);
            }
            out = deadv[j] ? stuck[c] : y;                                // Eq. 28 (D5 when l = u = 0)
          }
          if (ft_noisy) ft_noisy[ej * 6 + c] = out;
        }
      }
      if (delay_on) {  // keep the last Delta + J fields of the episode
        o.hist[e].push_back(cfield);
        while ((int)o.hist[e].size() > pr.read_delay + pr.read_jitter) o.hist[e].pop_front();
      }
    }
    // R10: noisy readouts of the scalar sensors (ContactDepth, Proximity, Elastomer markers): Table 3 gives them every
    // knob of App. A.8 except crosstalk.  Probe-level draws (gain stream 3, dead stream 2) are those of the taxel;
    // markers are probes of their own, numbered 0x80000000 + m in the taxel word of the counter.
    if (pr.noise_enable && (o.depth_noisy || o.prox_noisy || o.marker_noisy)) {
      const uint32_t n = o.n_step[e], ep4 = o.episode[e] << 4, env = (uint32_t)o.env_id[e];
      const uint32_t key[2] = {pr.seed_lo, pr.seed_hi};
      const uint32_t thr = (uint32_t)std::floor((double)pr.p_dead * 4294967296.0);
      const double decay = std::exp(-(double)pr.dt / (double)pr.tau);
      const bool gain_on = pr.gain_min != 1.0f || pr.gain_max != 1.0f;
      auto draw = [&](uint32_t probe, uint32_t step, uint32_t stream, uint32_t w[4]) {
        uint32_t c[4] = {env, probe, step, ep4 | stream};
        philox4x32_10(c, key, w);
      };
      // Read delay of the scalar readouts (Table 3: every sensor has it): the SAME Delta_n as the force / torque readout
      // of this env and step (one sensor read; stream 9, R9), applied to the post-hysteresis signal of each probe.
      const bool sdelay_on = pr.read_delay > 0 || pr.read_jitter > 0;
      int sdelta = 0;
      std::vector<double> scur;
      const double szero = 0.0;
      if (sdelay_on) {
        int k_n = 0;
        if (pr.read_jitter > 0) {
          uint32_t wj[4];
          draw(0xffffffffu, n, 9u, wj);
          k_n = (int)(((uint64_t)(wj[0] >> 9) * (uint64_t)(2 * pr.read_jitter + 1)) >> 23) - pr.read_jitter;
        }
        sdelta = std::max(0, pr.read_delay + k_n);
        scur.assign((size_t)T * 2 + (size_t)M * 3, 0.0);
      }
      const int shave = (int)o.shist[e].size();
      auto delayed_of = [&](size_t idx) -> const double* {   // the signal of step n - Delta_n, 0 before the episode began (Q12)
        if (!sdelay_on || sdelta == 0) return nullptr;
        return sdelta <= shave ? &o.shist[e][shave - sdelta][idx] : &szero;
      };
      for (int j = 0; j < T; ++j) {
        size_t ej = (size_t)e * T + j;
        double od = 0.0, op = 0.0;
        if (o.aux_sq_depth) o.aux_sq_depth[ej] = INFINITY;
        if (o.aux_sq_prox) o.aux_sq_prox[ej] = INFINITY;
        if (o.radius[j] > 0.0) {
          uint32_t w[4], ws[4], wg[4];
          draw((uint32_t)j, n, 10u, w);                          // stream 10: (0,1) -> depth (rw, white), (2,3) -> prox
          double zd[2], zp[2];
          box_muller(w[0], w[1], &zd[0], &zd[1]);
          box_muller(w[2], w[3], &zp[0], &zp[1]);
          draw((uint32_t)j, 0u, 11u, ws);                        // stream 11, n = 0: stuck values (word 0 depth, 1 prox)
          double gain = 1.0;
          if (gain_on) { draw((uint32_t)j, 0u, 3u, wg); gain = (double)pr.gain_min + ((double)pr.gain_max - (double)pr.gain_min) * word_to_uniform(wg[0]); }
          od = scalar_chain(pr, 0, dep_t[j], gain, deadv[j], word_to_uniform(ws[0]), zd[0], zd[1], o.sn_ha[ej * 2], o.sn_hb[ej * 2],
                            o.sn_dr[ej * 2], decay, o.aux_sq_depth ? &o.aux_sq_depth[ej] : nullptr, nullptr, delayed_of((size_t)j * 2),
                            sdelay_on ? &scur[(size_t)j * 2] : nullptr);
          op = scalar_chain(pr, 1, prox_c[j], gain, deadv[j], word_to_uniform(ws[1]), zp[0], zp[1], o.sn_ha[ej * 2 + 1],
                            o.sn_hb[ej * 2 + 1], o.sn_dr[ej * 2 + 1], decay, o.aux_sq_prox ? &o.aux_sq_prox[ej] : nullptr, nullptr,
                            delayed_of((size_t)j * 2 + 1), sdelay_on ? &scur[(size_t)j * 2 + 1] : nullptr);
        }
        if (o.depth_noisy) o.depth_noisy[ej] = od;
        if (o.prox_noisy) o.prox_noisy[ej] = op;
      }
      if (o.marker_noisy) {
        for (int jm = 0; jm < M; ++jm) {
          const int pm = o.mpatch[jm];
          const bool mact = o.radius[o.p_start[pm]] > 0.0;       // markers of a filtered-out link are fillers too
          const uint32_t probe = 0x80000000u + (uint32_t)jm;
          uint32_t w0[4], w1[4], wd[4], wg[4], ws[4];
          double zr[4] = {0, 0, 0, 0}, zw[2] = {0, 0};
          bool mdead = false;
          double gain = 1.0;
          if (mact) {
            draw(probe, n, 0u, w0);                              // stream 0: (0,1) -> rw ch 0,1; (2,3) -> rw ch 2, white ch 0
            draw(probe, n, 1u, w1);                              // stream 1: (0,1) -> white ch 1, 2
            box_muller(w0[0], w0[1], &zr[0], &zr[1]);
            box_muller(w0[2], w0[3], &zr[2], &zr[3]);
            box_muller(w1[0], w1[1], &zw[0], &zw[1]);
            draw(probe, 0u, 2u, wd);
            mdead = wd[0] < thr;
            if (gain_on) { draw(probe, 0u, 3u, wg); gain = (double)pr.gain_min + ((double)pr.gain_max - (double)pr.gain_min) * word_to_uniform(wg[0]); }
            draw(probe, 0u, 4u, ws);                             // stream 4, n = 0: stuck values, words 0-2
          }
          for (int c = 0; c < 3; ++c) {
            size_t i3 = ((size_t)e * M + jm) * 3 + c;
            double out = 0.0;
            if (o.aux_sq_marker) o.aux_sq_marker[i3] = INFINITY;
            if (o.aux_sasym_marker) o.aux_sasym_marker[i3] = INFINITY;
            if (mact)
              out = scalar_chain(pr, 2, marker_c[(size_t)jm * 3 + c], gain, mdead, word_to_uniform(ws[c]), zr[c],
                                 c == 0 ? zr[3] : zw[c - 1], o.sm_ha[i3], o.sm_hb[i3], o.sm_dr[i3], decay,
                                 o.aux_sq_marker ? &o.aux_sq_marker[i3] : nullptr, o.aux_sasym_marker ? &o.aux_sasym_marker[i3] : nullptr,
                                 delayed_of((size_t)T * 2 + (size_t)jm * 3 + c), sdelay_on ? &scur[(size_t)T * 2 + (size_t)jm * 3 + c] : nullptr);
            o.marker_noisy[i3] = out;
          }
        }
      }
      if (sdelay_on) {  // keep the last Delta + J signal fields of the episode
        o.shist[e].push_back(scur);
        while ((int)o.shist[e].size() > pr.read_delay + pr.read_jitter) o.shist[e].pop_front();
      }
    }
    o.n_step[e] += 1;
  }
}

// Comparator aid: aux_quant[E,T,6] receives, on every following step, the distance (in units of the
// readout) of the pre-quantisation value from the nearest rounding boundary of Eq. 25's quantize(),
// +inf where quantisation is off.  NULL switches it off.
void orc_set_aux_quant(void* h, double* aux_quant) { ((Oracle*)h)->aux_quant = aux_quant; }

// Comparator aid: aux_rgate[E,T] receives |R~_j - phi| (the distance of the perturbed d~ > 0 gate of Eq. 26,
// R8), +inf where radius noise is off or the slot is inactive.  NULL switches it off.
void orc_set_aux_rgate(void* h, double* aux_rgate) { ((Oracle*)h)->aux_rgate = aux_rgate; }

// Comparator aid: aux_wingap[E,T] receives phi_second - phi_best over the K objects of the env (the margin by
// which Eq. 2's winner g* won), +inf with fewer than two objects.  NULL switches it off.
void orc_set_aux_wingap(void* h, double* aux_wingap) { ((Oracle*)h)->aux_wingap = aux_wingap; }

// A.6: bank of tracked surface point clouds [n_clouds, n_points, 3] (object frame, fp32, copied) and the cloud of each
// (env, object) (-1 = not tracked); orc_set_proxpc hands in the [E,T,6] output the following orc_step calls fill.
int orc_set_pointclouds(void* h, int n_clouds, int n_points, const float* pts, const int32_t* cloud_id) {
  Oracle& o = *(Oracle*)h;
  o.pc_G = n_clouds; o.pc_N = n_points;
  o.pc_pts.assign(pts, pts + (size_t)n_clouds * n_points * 3);
  o.pc_id.assign(cloud_id, cloud_id + (size_t)o.E * o.K);
  for (int32_t id : o.pc_id) if (id >= n_clouds) return 1;
  size_t ns = (size_t)o.E * o.P * o.K * n_points;
  o.sh_on.assign(ns, 0); o.sh_e.assign(ns, V3{0, 0, 0});
  return 0;
}
void orc_set_proxpc(void* h, double* proxpc) { ((Oracle*)h)->proxpc = proxpc; }

// A.1 raycast backend: bank of triangle meshes (object frame; vertex / triangle offsets [n_meshes + 1]) and the mesh of
// each (env, object) (-1 = none); orc_set_raycast_out hands in the outputs of the following orc_step calls.
int orc_set_meshes(void* h, int n_meshes, const int32_t* vert_off, const int32_t* tri_off, const float* verts,
                   const int32_t* tris, const int32_t* mesh_id) {
  Oracle& o = *(Oracle*)h;
  o.rc_voff.assign(vert_off, vert_off + n_meshes + 1); o.rc_toff.assign(tri_off, tri_off + n_meshes + 1);
  o.rc_verts.assign(verts, verts + (size_t)vert_off[n_meshes] * 3);
  o.rc_tris.assign(tris, tris + (size_t)tri_off[n_meshes] * 3);
  o.rc_id.assign(mesh_id, mesh_id + (size_t)o.E * o.K);
  for (int32_t id : o.rc_id) if (id >= n_meshes) return 1;
  return 0;
}
void orc_set_raycast_out(void* h, double* depth, double* nrm, double* gap) {
  Oracle& o = *(Oracle*)h;
  o.rc_depth = depth; o.rc_nrm = nrm; o.rc_gap = gap;
}
void orc_closest_point_triangle(const double* p, const double* a, const double* b, const double* c, double* out) {
  V3 r = closest_point_triangle({p[0], p[1], p[2]}, {a[0], a[1], a[2]}, {b[0], b[1], b[2]}, {c[0], c[1], c[2]});
  out[0] = r.x; out[1] = r.y; out[2] = r.z;
}
double orc_ray_triangle(const double* o, const double* d, const double* a, const double* b, const double* c) {
  return ray_triangle({o[0], o[1], o[2]}, {d[0], d[1], d[2]}, {a[0], a[1], a[2]}, {b[0], b[1], b[2]}, {c[0], c[1], c[2]});
}

// R10: hands in the buffers the following orc_step calls fill with the noisy scalar readouts (NULL = not produced) and
// their comparator aids (distance to the quantisation boundary per element; marker ASYM sign-flip margin).
void orc_set_scalar_noisy(void* h, double* depth_noisy, double* prox_noisy, double* marker_noisy, double* aux_sq_depth,
                          double* aux_sq_prox, double* aux_sq_marker, double* aux_sasym_marker) {
  Oracle& o = *(Oracle*)h;
  o.depth_noisy = depth_noisy; o.prox_noisy = prox_noisy; o.marker_noisy = marker_noisy;
  o.aux_sq_depth = aux_sq_depth; o.aux_sq_prox = aux_sq_prox; o.aux_sq_marker = aux_sq_marker; o.aux_sasym_marker = aux_sasym_marker;
}

// Stand-alone pieces for the pins -------------------------------------------------

// O5 on explicit arguments (all double[3] except quat float[4]); out[6].
void orc_kinematic_ft(const orc_params* pr, double d, const double* m_world, const double* x_j, const float* quat_L,
                      const double* pL, const double* vL, const double* wL, const double* pO, const double* vO,
                      const double* wO, double* out) {
  M3 RL = quat_to_R(quat_L);
  V3 xj = {x_j[0], x_j[1], x_j[2]};
  V3 pl = {pL[0], pL[1], pL[2]};
  V3 q = pl + mul(RL, xj);
  kinematic_ft(*pr, d, {m_world[0], m_world[1], m_world[2]}, q, xj, RL, pl, {vL[0], vL[1], vL[2]}, {wL[0], wL[1], wL[2]},
               {pO[0], pO[1], pO[2]}, {vO[0], vO[1], vO[2]}, {wO[0], wO[1], wO[2]}, out);
}

// O7 on one geometry in its own frame: start x0, direction a (object frame).
double orc_march(int type, const double* params, const float* grid, int N, double hv, const double* x0, const double* a,
                 double r_prox, int steps) {
  Geom g; g.type = type; for (int i = 0; i < 4; ++i) g.p[i] = params ? params[i] : 0.0;
  g.grid = grid; g.N = N; g.hv = hv;
  V3 x = {x0[0], x0[1], x0[2]}, d = {a[0], a[1], a[2]};
  return march([&](double t) { return sdf_eval(g, x + t * d).phi; }, r_prox, steps);
}

int orc_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
