// Hand-written sm_100a kernels of the batched tactile readout.  Citations: "P:NNN" = line of
// the paper text (App. A = P:172-359); "D*/Q*/O*" = readings listed in DESIGN.md.
//
// Mapping: ONE WARP PER (environment, patch).  A patch has <= 64 taxel slots; lane l owns the
// two consecutive slots i = 2l and 2l+1 (so every per-taxel stream is read/written as one
// 8-, 16- or 48-byte vector per lane) and the two markers l and l+32.  The link pose, the
// link->object transform and the velocity terms are warp-uniform; crosstalk neighbours are
// fetched with __shfl_sync, marker sources are broadcast with __shfl_sync.
//
// Bank layout ("quad"): for every grid, Q[(j*(N-1) + i)*N + k] = float4(phi(i,j,k), phi(i+1,j,k),
// phi(i,j+1,k), phi(i+1,j+1,k)), i,j in [0,N-2], k in [0,N-1].  The 8 corners of cell (i,j,k) are
// the two consecutive float4 Q[..k], Q[..k+1]: one 32-byte span, two LDG.128 instead of eight
// scattered LDG.32 (the L1 wavefront count of the gather is what bounds the SDF path).
#include <cuda_runtime.h>

#include <cstdint>

#include "ts_internal.h"

#define TS_BLOCK 128

namespace {

struct F3 {
  float x, y, z;
};
__device__ __forceinline__ F3 mk3(float x, float y, float z) { return F3{x, y, z}; }
__device__ __forceinline__ F3 operator+(F3 a, F3 b) { return F3{a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ F3 operator-(F3 a, F3 b) { return F3{a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ F3 operator*(float s, F3 a) { return F3{s * a.x, s * a.y, s * a.z}; }
__device__ __forceinline__ float dot(F3 a, F3 b) { return fmaf(a.x, b.x, fmaf(a.y, b.y, a.z * b.z)); }
__device__ __forceinline__ F3 cross(F3 a, F3 b) {
  return F3{a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x};
}
__device__ __forceinline__ F3 ld3(const float* p) { return F3{__ldg(p), __ldg(p + 1), __ldg(p + 2)}; }

struct Rot {  // row-major 3x3
  float a[9];
};
__device__ __forceinline__ F3 mul(const Rot& R, F3 v) {
  return F3{fmaf(R.a[0], v.x, fmaf(R.a[1], v.y, R.a[2] * v.z)), fmaf(R.a[3], v.x, fmaf(R.a[4], v.y, R.a[5] * v.z)),
            fmaf(R.a[6], v.x, fmaf(R.a[7], v.y, R.a[8] * v.z))};
}
__device__ __forceinline__ F3 mulT(const Rot& R, F3 v) {
  return F3{fmaf(R.a[0], v.x, fmaf(R.a[3], v.y, R.a[6] * v.z)), fmaf(R.a[1], v.x, fmaf(R.a[4], v.y, R.a[7] * v.z)),
            fmaf(R.a[2], v.x, fmaf(R.a[5], v.y, R.a[8] * v.z))};
}

// Double-precision twins used ONLY for the relative pose and the first geometry query (DESIGN.md
// "fp64 frame"): the contact normal of a box edge/corner is max(|x|-b,0)/|.|, a ratio of
// millimetre differences of centimetre numbers, and the stiff force law amplifies d; with fp32
// positions (error ~4e-9 m) neither meets rtol 1e-4.  B200 issues DFMA at half the FFMA rate
// and this is ~60 DFMA per taxel, so the cost hides under the state streams.
template <typename S>
struct X3 {
  S x, y, z;
};
typedef X3<double> D3;
struct RotD {
  double a[9];
};
// O0: rotation of a quaternion (w,x,y,z), used as given.
__device__ __forceinline__ RotD quat_Rd(const float* q4) {
  const float4 q = __ldg(reinterpret_cast<const float4*>(q4));
  const double w = q.x, x = q.y, y = q.z, z = q.w;
  RotD R;
  R.a[0] = 1.0 - 2.0 * (y * y + z * z); R.a[1] = 2.0 * (x * y - w * z);       R.a[2] = 2.0 * (x * z + w * y);
  R.a[3] = 2.0 * (x * y + w * z);       R.a[4] = 1.0 - 2.0 * (x * x + z * z); R.a[5] = 2.0 * (y * z - w * x);
  R.a[6] = 2.0 * (x * z - w * y);       R.a[7] = 2.0 * (y * z + w * x);       R.a[8] = 1.0 - 2.0 * (x * x + y * y);
  return R;
}
__device__ __forceinline__ Rot to_float(const RotD& R) {
  Rot r;
#pragma unroll
  for (int i = 0; i < 9; ++i) r.a[i] = (float)R.a[i];
  return r;
}
__device__ __forceinline__ F3 to_float(const D3& v) { return F3{(float)v.x, (float)v.y, (float)v.z}; }
__device__ __forceinline__ X3<float> as_x3(F3 v) { return X3<float>{v.x, v.y, v.z}; }

// Object k seen from the sensor link: x_o = c + M x_j (object frame <- link frame).
// Forming p_L - p_O BEFORE rotating keeps the small relative offsets accurate.
struct ObjFrame {
  Rot M;  // R_O^T R_L
  F3 c;   // R_O^T (p_L - p_O)
  int type;
  float4 prm;
};
struct ObjFrameD {
  RotD M;
  D3 c;
};

__device__ __forceinline__ ObjFrame make_frame(const TsStepParams& p, int e, int k, const RotD& RL, D3 pL, ObjFrameD& fd) {
  const size_t ek = (size_t)e * p.K + k;
  ObjFrame f;
  f.type = __ldg(p.g_type + ek);
  f.prm = __ldg(p.g_params + ek);
  const RotD RO = quat_Rd(p.obj_quat + ek * 4);
  const double dx = pL.x - (double)__ldg(p.obj_pos + ek * 3), dy = pL.y - (double)__ldg(p.obj_pos + ek * 3 + 1),
               dz = pL.z - (double)__ldg(p.obj_pos + ek * 3 + 2);
#pragma unroll
  for (int r = 0; r < 3; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c)
      fd.M.a[r * 3 + c] = fma(RO.a[r], RL.a[c], fma(RO.a[3 + r], RL.a[3 + c], RO.a[6 + r] * RL.a[6 + c]));
  fd.c.x = fma(RO.a[0], dx, fma(RO.a[3], dy, RO.a[6] * dz));
  fd.c.y = fma(RO.a[1], dx, fma(RO.a[4], dy, RO.a[7] * dz));
  fd.c.z = fma(RO.a[2], dx, fma(RO.a[5], dy, RO.a[8] * dz));
  f.M = to_float(fd.M);
  f.c = to_float(fd.c);
  return f;
}
__device__ __forceinline__ D3 mul(const ObjFrameD& f, F3 v) {
  const double x = v.x, y = v.y, z = v.z;
  return D3{fma(f.M.a[0], x, fma(f.M.a[1], y, fma(f.M.a[2], z, f.c.x))), fma(f.M.a[3], x, fma(f.M.a[4], y, fma(f.M.a[5], z, f.c.y))),
            fma(f.M.a[6], x, fma(f.M.a[7], y, fma(f.M.a[8], z, f.c.z)))};
}

// ---------------------------------------------------------------------------------------
// O2: signed distance (and object-frame gradient) of one geometry at object-frame point x.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ float inv_vox(const TsStepParams& p, float) { return p.inv_voxel; }
__device__ __forceinline__ double inv_vox(const TsStepParams& p, double) { return p.inv_voxel_d; }
__device__ __forceinline__ float fma_s(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double fma_s(double a, double b, double c) { return fma(a, b, c); }

// S = double for the first query (cell index and fractions exact to fp32 rounding), float in the march.
template <bool GRAD, typename S>
__device__ __forceinline__ float sdf_grid(const TsStepParams& p, int gid, X3<S> x, F3& g) {
  const int N = p.grid_n;
  const S top = (S)(N - 1);
  const S half = (S)0.5 * top;
  const S iv = inv_vox(p, S());
  const S ux = fma_s(x.x, iv, half), uy = fma_s(x.y, iv, half), uz = fma_s(x.z, iv, half);
  const S cx = min(max(ux, (S)0), top), cy = min(max(uy, (S)0), top), cz = min(max(uz, (S)0), top);
  const int i0 = min((int)cx, N - 2), j0 = min((int)cy, N - 2), k0 = min((int)cz, N - 2);
  const float fx = (float)(cx - (S)i0), fy = (float)(cy - (S)j0), fz = (float)(cz - (S)k0);
  const float4* q = p.bank + (size_t)gid * p.grid_stride + ((size_t)(j0 * (N - 1) + i0) * N + k0);
  const float4 A = __ldg(q), B = __ldg(q + 1);  // (c000,c100,c010,c110), (c001,c101,c011,c111)
  const float a0 = fmaf(fx, A.y - A.x, A.x), a1 = fmaf(fx, A.w - A.z, A.z);
  const float b0 = fmaf(fx, B.y - B.x, B.x), b1 = fmaf(fx, B.w - B.z, B.z);
  const float lo = fmaf(fy, a1 - a0, a0), hi = fmaf(fy, b1 - b0, b0);
  float phi = fmaf(fz, hi - lo, lo);
  const float ox = (float)(ux - cx), oy = (float)(uy - cy), oz = (float)(uz - cz);   // outside-grid extension (O2)
  const float o2 = fmaf(ox, ox, fmaf(oy, oy, oz * oz));
  if (o2 > 0.f) phi += p.voxel * sqrtf(o2);
  if (GRAD) {  // exact derivative of the trilinear interpolant in cell (i0,j0,k0); 1/h_v dropped (normalised later)
    const float gy0 = 1.f - fy, gz0 = 1.f - fz;
    const float dxa = fmaf(fy, A.w - A.z, gy0 * (A.y - A.x)), dxb = fmaf(fy, B.w - B.z, gy0 * (B.y - B.x));
    g.x = fmaf(fz, dxb, gz0 * dxa);
    g.y = fmaf(fz, b1 - b0, gz0 * (a1 - a0));
    g.z = hi - lo;
  }
  return phi;
}

template <bool GRAD, typename S>
__device__ __forceinline__ float sdf_eval(const TsStepParams& p, const ObjFrame& f, X3<S> xs, F3& g) {
  const F3 x = mk3((float)xs.x, (float)xs.y, (float)xs.z);
  switch (f.type) {
    case TS_GEOM_SPHERE: {
      const float n = sqrtf(dot(x, x));
      if (GRAD) g = (n < 1e-12f) ? mk3(0.f, 0.f, 1.f) : (1.f / n) * x;
      return n - f.prm.x;
    }
    case TS_GEOM_BOX: {  // w = |x| - b formed in S: the edge/corner normal is a ratio of these small differences
      const float wx = (float)(abs(xs.x) - (S)f.prm.x), wy = (float)(abs(xs.y) - (S)f.prm.y), wz = (float)(abs(xs.z) - (S)f.prm.z);
      const float px = fmaxf(wx, 0.f), py = fmaxf(wy, 0.f), pz = fmaxf(wz, 0.f);
      const float lp = sqrtf(fmaf(px, px, fmaf(py, py, pz * pz)));
      const float wmax = fmaxf(wx, fmaxf(wy, wz));
      if (GRAD) {
        const float sx = x.x < 0.f ? -1.f : 1.f, sy = x.y < 0.f ? -1.f : 1.f, sz = x.z < 0.f ? -1.f : 1.f;
        if (wmax > 0.f) {
          const float il = 1.f / lp;
          g = mk3(sx * px * il, sy * py * il, sz * pz * il);
        } else {  // interior: axis of the largest w, ties -> lowest index (Q7)
          g = mk3(0.f, 0.f, 0.f);
          if (wx >= wy && wx >= wz) g.x = sx;
          else if (wy >= wz) g.y = sy;
          else g.z = sz;
        }
      }
      return lp + fminf(wmax, 0.f);
    }
    case TS_GEOM_CAPSULE: {
      const float zc = fminf(fmaxf(x.z, -f.prm.y), f.prm.y);
      const F3 y = mk3(x.x, x.y, x.z - zc);
      const float n = sqrtf(dot(y, y));
      if (GRAD) g = (n < 1e-12f) ? mk3(0.f, 0.f, 1.f) : (1.f / n) * y;
      return n - f.prm.x;
    }
    case TS_GEOM_SDF:
      return sdf_grid<GRAD, S>(p, (int)f.prm.x, xs, g);
    default:
      if (GRAD) g = mk3(0.f, 0.f, 1.f);
      return __int_as_float(0x7f800000);
  }
}

// ---------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al. 2011), counter = (env, taxel, n, episode<<4 | stream) (O8).
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
    c = make_uint4(hi1 ^ c.y ^ k0, lo1, hi0 ^ c.w ^ k1, lo0);
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  return c;
}
// u = (2 (w >> 9) + 1) 2^-24: exact in fp32, never 0 or 1.
__device__ __forceinline__ float u01(uint32_t w) { return (float)(2u * (w >> 9) + 1u) * 5.9604644775390625e-8f; }
__device__ __forceinline__ void box_muller(uint32_t wa, uint32_t wb, float& z0, float& z1) {
  const float r = sqrtf(-2.f * logf(u01(wa)));
  float s, c;
  sincospif(2.f * u01(wb), &s, &c);  // 2 u_b is exact; sin/cos(2 pi u_b)
  z0 = r * c;
  z1 = r * s;
}

__device__ __forceinline__ void st_stream(float* p, float v) { __stcs(p, v); }

// ---------------------------------------------------------------------------------------
// The fused step kernel: S1-S8 of DESIGN.md for one (env, patch) per warp.
// ---------------------------------------------------------------------------------------
template <bool SINGLE>
__global__ void __launch_bounds__(TS_BLOCK) ts_step_kernel(const __grid_constant__ TsStepParams p) {
  const int lane = threadIdx.x & 31;
  const long long gw = ((long long)blockIdx.x * TS_BLOCK + threadIdx.x) >> 5;
  if (gw >= (long long)p.E * p.P) return;
  const int e = (int)(gw / p.P);
  const int pi = (int)(gw - (long long)e * p.P);
  const int4 pa = __ldg(reinterpret_cast<const int4*>(p.patches + pi));
  const int4 pb = __ldg(reinterpret_cast<const int4*>(p.patches + pi) + 1);
  const int start = pa.x, n = pa.y, nu = pa.z, link = pa.w, mstart = pb.x, mcount = pb.y;
  const float eps = __int_as_float(pb.z);
  const size_t eT = (size_t)e * p.T;
  const int i0 = 2 * lane;
  const size_t j0 = eT + start + i0;  // global slot of my first taxel
  bool valid[2] = {i0 < n, i0 + 1 < n};
  const bool vec_ok = valid[1] && ((j0 & 1) == 0);  // both slots present and the pair is 8/16-byte aligned

  // ---- per-taxel layout (shared by all envs; L1/L2 resident) --------------------------
  F3 xj[2], nj[2];
  float Rj[2];
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    const int t = start + min(i0 + s, n - 1);
    const float4 a = __ldg(p.tx_pos + t), b = __ldg(p.tx_nrm + t);
    xj[s] = mk3(a.x, a.y, a.z);
    nj[s] = mk3(b.x, b.y, b.z);
    Rj[s] = (valid[s] && link >= 0) ? a.w : 0.f;  // R_j = 0: inactive filler
  }
  const bool act[2] = {Rj[0] > 0.f, Rj[1] > 0.f};

  // ---- S1: link pose (warp-uniform) ---------------------------------------------------
  const int lk = max(link, 0);
  const size_t el = (size_t)e * p.L + lk;
  const RotD RLd = quat_Rd(p.link_quat + el * 4);
  const Rot RL = to_float(RLd);
  const F3 pL = ld3(p.link_pos + el * 3);
  const D3 pLd = D3{(double)pL.x, (double)pL.y, (double)pL.z};

  // ---- S2/S3: geometry query, winner = smallest phi (= max_k [R - phi_k]_+, Eq. 2) ------
  ObjFrameD frd;
  ObjFrame fr = make_frame(p, e, 0, RLd, pLd, frd);
  float phi[2];
  F3 mbar[2];  // contact normal in the link frame, m_bar = R_L^T m = M^T g/|g|
  int kst[2] = {0, 0};
  F3 xo[2], dro[2];  // object-frame taxel position and march direction (SINGLE only)
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    phi[s] = __int_as_float(0x7f800000);
    mbar[s] = mk3(0.f, 0.f, 0.f);
  }
  for (int k = 0; k < (SINGLE ? 1 : p.K); ++k) {
    if (!SINGLE && k > 0) fr = make_frame(p, e, k, RLd, pLd, frd);
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      const D3 xd = mul(frd, xj[s]);
      if (SINGLE) { xo[s] = to_float(xd); dro[s] = mul(fr.M, nj[s]); }
      F3 g;
      const float ph = sdf_eval<true, double>(p, fr, xd, g);
      if (ph < phi[s]) {  // strict: ties -> lowest k (Q3)
        phi[s] = ph;
        kst[s] = k;
        const float gn = sqrtf(dot(g, g));
        mbar[s] = (gn < 1e-12f) ? (-1.f) * nj[s] : (1.f / gn) * mulT(fr.M, g);  // Q2
      }
    }
  }

  // ---- S4: depth (Eq. 2) and Schmitt contact bit (Eq. 3) ------------------------------
  float d[2];
  uint8_t flag[2];
  {
    uchar2 fl = make_uchar2(0, 0);
    if (vec_ok) fl = *reinterpret_cast<const uchar2*>(p.st_flags + j0);
    else { if (valid[0]) fl.x = p.st_flags[j0]; if (valid[1]) fl.y = p.st_flags[j0 + 1]; }
    flag[0] = fl.x; flag[1] = fl.y;
  }
  uint8_t yb[2], deadb[2];
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    d[s] = act[s] ? fmaxf(0.f, Rj[s] - phi[s]) : 0.f;
    const bool y = act[s] && ((d[s] > p.eta_on) || ((flag[s] & 1) && d[s] > p.eta_off));
    deadb[s] = (p.noise_enable && act[s]) ? ((flag[s] >> 1) & 1) : 0;
    yb[s] = y ? 1 : 0;
    flag[s] = (flag[s] & 2) | yb[s];
  }
  if (vec_ok) {
    *reinterpret_cast<uchar2*>(p.st_flags + j0) = make_uchar2(flag[0], flag[1]);
    if (p.contact) *reinterpret_cast<uchar2*>(p.contact + j0) = make_uchar2(deadb[0] ? 0 : yb[0], deadb[1] ? 0 : yb[1]);
    if (p.dead) *reinterpret_cast<uchar2*>(p.dead + j0) = make_uchar2(deadb[0], deadb[1]);
    if (p.depth) __stcs(reinterpret_cast<float2*>(p.depth + j0), make_float2(d[0], d[1]));
  } else {
#pragma unroll
    for (int s = 0; s < 2; ++s)
      if (valid[s]) {
        p.st_flags[j0 + s] = flag[s];
        if (p.contact) p.contact[j0 + s] = deadb[s] ? 0 : yb[s];
        if (p.dead) p.dead[j0 + s] = deadb[s];
        if (p.depth) st_stream(p.depth + j0 + s, d[s]);
      }
  }

  // ---- S5: kinematic force / torque (Eq. 4-9, D2), link frame -------------------------
  float ft[2][6];
#pragma unroll
  for (int s = 0; s < 2; ++s)
#pragma unroll
    for (int c = 0; c < 6; ++c) ft[s][c] = 0.f;
  const bool want_ft = (p.ft != nullptr) || p.noise_enable;
  if (want_ft && __any_sync(0xffffffffu, d[0] > 0.f || d[1] > 0.f)) {
    // link-frame velocity terms: v_rel = vbar + wO x (cbar + x_j) - wL x x_j
    const F3 vL = ld3(p.link_linvel + el * 3), wLw = ld3(p.link_angvel + el * 3);
    const F3 wL = mulT(RL, wLw);
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      if (d[s] > 0.f) {  // Q5: every term gated on d > 0
        const size_t ek = (size_t)e * p.K + kst[s];
        const float sj = __powf(d[s], p.alpha);  // s_j = d^alpha
        F3 f, tau;
        if (p.use_velocity) {
          const F3 pO = ld3(p.obj_pos + ek * 3), vO = ld3(p.obj_linvel + ek * 3), wOw = ld3(p.obj_angvel + ek * 3);
          const F3 wO = mulT(RL, wOw), vbar = mulT(RL, vO - vL), cbar = mulT(RL, pL - pO);
          const F3 vrel = vbar + cross(wO, cbar + xj[s]) - cross(wL, xj[s]);           // Eq. 4-6
          const float vns = dot(vrel, mbar[s]);
          const F3 vt = vrel - vns * mbar[s];                                          // Eq. 7
          const F3 fn = (sj * fmaf(p.c_n, vns, p.k_n)) * mbar[s];                      // Eq. 8 normal
          F3 ftan = (-p.k_t) * vt;                                                     // Eq. 8 tangential
          const float lim = p.mu * sqrtf(dot(fn, fn)), nft = sqrtf(dot(ftan, ftan));
          if (nft > lim) ftan = (lim / nft) * ftan;                                    // D2 Coulomb cap
          f = fn + ftan;
          tau = cross(xj[s], f) - (p.k_omega * dot(wO - wL, mbar[s])) * mbar[s];       // Eq. 9
        } else {
          f = (p.k_n * sj) * mbar[s];
          tau = cross(xj[s], f);
        }
        ft[s][0] = f.x; ft[s][1] = f.y; ft[s][2] = f.z; ft[s][3] = tau.x; ft[s][4] = tau.y; ft[s][5] = tau.z;
      }
    }
  }
  if (p.ft) {
    float* o = p.ft + j0 * 6;
    if (vec_ok) {
      __stcs(reinterpret_cast<float4*>(o), make_float4(ft[0][0], ft[0][1], ft[0][2], ft[0][3]));
      __stcs(reinterpret_cast<float4*>(o) + 1, make_float4(ft[0][4], ft[0][5], ft[1][0], ft[1][1]));
      __stcs(reinterpret_cast<float4*>(o) + 2, make_float4(ft[1][2], ft[1][3], ft[1][4], ft[1][5]));
    } else {
#pragma unroll
      for (int s = 0; s < 2; ++s)
        if (valid[s])
#pragma unroll
          for (int c = 0; c < 6; ++c) st_stream(o + s * 6 + c, ft[s][c]);
    }
  }

  // ---- S8: noise chain on the six channels (O8): hysteresis -> crosstalk -> drift -> dead
  if (p.noise_enable) {
    const size_t blk = (size_t)e * p.P + pi;
    float h[2][6];
    // S8b hysteresis; state rows are [row][lane] float4 so each load is one 512-byte warp transaction
    if (p.hyst_mode == TS_HYST_ASYM) {
      float4* st = p.st_hyst + blk * (3 * 32) + lane;
      float y[12];
      if (valid[0]) {
#pragma unroll
        for (int r = 0; r < 3; ++r) {
          const float4 v = __ldcs(st + r * 32);
          y[4 * r] = v.x; y[4 * r + 1] = v.y; y[4 * r + 2] = v.z; y[4 * r + 3] = v.w;
        }
      } else {
#pragma unroll
        for (int i = 0; i < 12; ++i) y[i] = 0.f;
      }
#pragma unroll
      for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int c = 0; c < 6; ++c) {
          const float x = ft[s][c], yp = y[s * 6 + c];
          const float al = (fabsf(x) > fabsf(yp)) ? p.alpha_load : p.alpha_unload;  // D3, Q14
          const float yn = act[s] ? fmaf(al, x - yp, yp) : 0.f;
          y[s * 6 + c] = yn;
          h[s][c] = yn;
        }
      if (valid[0]) {
#pragma unroll
        for (int r = 0; r < 3; ++r) __stcs(st + r * 32, make_float4(y[4 * r], y[4 * r + 1], y[4 * r + 2], y[4 * r + 3]));
      }
    } else if (p.hyst_mode == TS_HYST_MAXWELL) {
      float4* st = p.st_hyst + blk * (6 * 32) + lane;
      float xi[12], xp[12];
      if (valid[0]) {
#pragma unroll
        for (int r = 0; r < 3; ++r) {
          const float4 v = __ldcs(st + r * 32), w = __ldcs(st + (3 + r) * 32);
          xi[4 * r] = v.x; xi[4 * r + 1] = v.y; xi[4 * r + 2] = v.z; xi[4 * r + 3] = v.w;
          xp[4 * r] = w.x; xp[4 * r + 1] = w.y; xp[4 * r + 2] = w.z; xp[4 * r + 3] = w.w;
        }
      } else {
#pragma unroll
        for (int i = 0; i < 12; ++i) { xi[i] = 0.f; xp[i] = 0.f; }
      }
#pragma unroll
      for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int c = 0; c < 6; ++c) {
          const float x = ft[s][c];
          const float z = act[s] ? fmaf(p.decay, xi[s * 6 + c], x - xp[s * 6 + c]) : 0.f;  // Eq. 29
          xi[s * 6 + c] = z;
          xp[s * 6 + c] = act[s] ? x : 0.f;
          h[s][c] = fmaf(p.beta, z, x);                                                    // Eq. 30
        }
      if (valid[0]) {
#pragma unroll
        for (int r = 0; r < 3; ++r) {
          __stcs(st + r * 32, make_float4(xi[4 * r], xi[4 * r + 1], xi[4 * r + 2], xi[4 * r + 3]));
          __stcs(st + (3 + r) * 32, make_float4(xp[4 * r], xp[4 * r + 1], xp[4 * r + 2], xp[4 * r + 3]));
        }
      }
    } else {
#pragma unroll
      for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int c = 0; c < 6; ++c) h[s][c] = ft[s][c];
    }

    // S8c crosstalk (D4): c_j = h_j + chi/4 sum_{k in N4(j)} (h_k - h_j), neighbours by shuffle.
    // Slot i = 2 lane + s sits at (iu, iv) = (i mod nu, i div nu); -u/+u neighbours are i-+1,
    // -v/+v neighbours are i-+nu, i.e. lane (i-+nu)>>1, slot (i-+nu)&1.
    float cx[2][6];
    {
      const int nv_ = n / nu;
      const bool odd = nu & 1;
      int iu[2], iv[2];
#pragma unroll
      for (int s = 0; s < 2; ++s) { iv[s] = (i0 + s) / nu; iu[s] = (i0 + s) - iv[s] * nu; }
      const float q = 0.25f * p.chi;
#pragma unroll
      for (int c = 0; c < 6; ++c) {
        const float up1 = __shfl_up_sync(0xffffffffu, h[1][c], 1);      // slot 1 of lane-1  = taxel i0-1
        const float dn0 = __shfl_down_sync(0xffffffffu, h[0][c], 1);    // slot 0 of lane+1  = taxel i0+2
        float acc0 = 0.f, acc1 = 0.f;
        if (iu[0] > 0) acc0 += up1 - h[0][c];
        if (iu[0] < nu - 1) acc0 += h[1][c] - h[0][c];
        if (iu[1] > 0) acc1 += h[0][c] - h[1][c];
        if (iu[1] < nu - 1) acc1 += dn0 - h[1][c];
#pragma unroll
        for (int s = 0; s < 2; ++s) {
          const int im = i0 + s - nu, ip = i0 + s + nu;
          // source slot is warp-uniform: same slot when nu is even, the other one when odd
          const float srcm = odd ? h[1 - s][c] : h[s][c];
          const float vm = __shfl_sync(0xffffffffu, srcm, (im >> 1) & 31);
          const float vp = __shfl_sync(0xffffffffu, srcm, (ip >> 1) & 31);
          float a = 0.f;
          if (iv[s] > 0) a += vm - h[s][c];
          if (iv[s] < nv_ - 1) a += vp - h[s][c];
          if (s == 0) acc0 += a; else acc1 += a;
        }
        cx[0][c] = fmaf(q, acc0, h[0][c]);
        cx[1][c] = fmaf(q, acc1, h[1][c]);
      }
    }

    // S8d drift (Eq. 25): D <- D + sigma z, z from Philox + Box-Muller; S8a dead (Eq. 28)
    {
      float4* st = p.st_drift + blk * (3 * 32) + lane;
      float D[12];
      if (valid[0]) {
#pragma unroll
        for (int r = 0; r < 3; ++r) {
          const float4 v = __ldcs(st + r * 32);
          D[4 * r] = v.x; D[4 * r + 1] = v.y; D[4 * r + 2] = v.z; D[4 * r + 3] = v.w;
        }
      } else {
#pragma unroll
        for (int i = 0; i < 12; ++i) D[i] = 0.f;
      }
      const uint32_t nstep = p.gstep - __ldg(p.reset_step + e);
      const uint32_t ep4 = __ldg(p.episode + e) << 4;
      const uint32_t env = p.env_id_base + (uint32_t)e;
      float outv[12];
#pragma unroll
      for (int s = 0; s < 2; ++s) {
        float z[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        if (act[s]) {
          const uint32_t tax = (uint32_t)(start + i0 + s);
          const uint4 w0 = philox4x32_10(make_uint4(env, tax, nstep, ep4 | 0u), p.seed_lo, p.seed_hi);
          const uint4 w1 = philox4x32_10(make_uint4(env, tax, nstep, ep4 | 1u), p.seed_lo, p.seed_hi);
          box_muller(w0.x, w0.y, z[0], z[1]);
          box_muller(w0.z, w0.w, z[2], z[3]);
          box_muller(w1.x, w1.y, z[4], z[5]);
        }
#pragma unroll
        for (int c = 0; c < 6; ++c) {
          const float Dn = act[s] ? fmaf(c < 3 ? p.sigma_f : p.sigma_t, z[c], D[s * 6 + c]) : 0.f;
          D[s * 6 + c] = Dn;
          outv[s * 6 + c] = (act[s] && !deadb[s]) ? cx[s][c] + Dn : 0.f;
        }
      }
      if (valid[0]) {
#pragma unroll
        for (int r = 0; r < 3; ++r) __stcs(st + r * 32, make_float4(D[4 * r], D[4 * r + 1], D[4 * r + 2], D[4 * r + 3]));
      }
      if (p.ft_noisy) {
        float* o = p.ft_noisy + j0 * 6;
        if (vec_ok) {
#pragma unroll
          for (int r = 0; r < 3; ++r)
            __stcs(reinterpret_cast<float4*>(o) + r, make_float4(outv[4 * r], outv[4 * r + 1], outv[4 * r + 2], outv[4 * r + 3]));
        } else {
#pragma unroll
          for (int s = 0; s < 2; ++s)
            if (valid[s])
#pragma unroll
              for (int c = 0; c < 6; ++c) st_stream(o + s * 6 + c, outv[s * 6 + c]);
        }
      }
    }
  }

  // ---- S6: elastomer marker dilation (Eq. 18-21; sources with h_i = 0 contribute exactly 0)
  if (p.marker && mcount > 0) {
    float hh[2], ha[2];
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      hh[s] = act[s] ? fmaxf(0.f, -phi[s]) : 0.f;                  // Eq. 19
      ha[s] = hh[s] > 0.f ? __powf(hh[s], p.alpha_e) : 0.f;
    }
    unsigned m0 = __ballot_sync(0xffffffffu, hh[0] > 0.f), m1 = __ballot_sync(0xffffffffu, hh[1] > 0.f);
    F3 acc[2] = {mk3(0.f, 0.f, 0.f), mk3(0.f, 0.f, 0.f)};
    F3 mp[2], mn[2];
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      const int jm = mstart + min(lane + 32 * r, mcount - 1);
      const float4 a = __ldg(p.mk_pos + jm), b = __ldg(p.mk_nrm + jm);
      mp[r] = mk3(a.x, a.y, a.z);
      mn[r] = mk3(b.x, b.y, b.z);
    }
    const float two_eps = 2.f * eps, eps2 = eps * eps, cg = p.c_e * p.inv_gbar, crho = 1.f - p.c_e;
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      unsigned m = s ? m1 : m0;
      while (m) {
        const int sl = __ffs(m) - 1;
        m &= m - 1;
        const float hi = __shfl_sync(0xffffffffu, hh[s], sl), hai = __shfl_sync(0xffffffffu, ha[s], sl);
        const float4 xs = __ldg(p.tx_pos + start + 2 * sl + s);  // uniform address: broadcast
#pragma unroll
        for (int r = 0; r < 2; ++r) {
          const F3 z = mp[r] - mk3(xs.x, xs.y, xs.z);
          const F3 rr = z - dot(z, mn[r]) * mn[r];                 // Eq. 18
          const float r2 = dot(rr, rr);
          const float g = __expf(-p.lambda_d * r2);
          float w = cg * g;
          if (crho != 0.f) w = fmaf(crho, __fdividef(two_eps, r2 + eps2), w);
          w *= hi;                                                 // Eq. 20
          acc[r] = acc[r] + p.s_d * (w * rr + (hai * g) * mn[r]);  // Eq. 21
        }
      }
    }
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      const int jm = lane + 32 * r;
      if (jm < mcount) {
        float* o = p.marker + ((size_t)e * p.M + mstart + jm) * 3;
        st_stream(o, acc[r].x); st_stream(o + 1, acc[r].y); st_stream(o + 2, acc[r].z);
      }
    }
  }

  // ---- S7: proximity march (O7): t <- min(t + max(phi(q + t a), 0), r_prox), K_m evaluations.
  // Exact shortcuts: evaluation 0 is the query above; t = r_prox is absorbing; an evaluation
  // that leaves t unchanged (s <= 0, or s below half an ulp of t) repeats forever.
  if (p.prox) {
    float t[2];
    bool go[2];
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      t[s] = 0.f;
      go[s] = false;
      if (act[s] && p.march_steps > 0) {
        t[s] = fminf(fmaxf(phi[s], 0.f), p.r_prox);
        go[s] = (t[s] > 0.f) && (t[s] < p.r_prox);
      }
    }
    for (int it = 1; it < p.march_steps; ++it) {
      if (!(go[0] || go[1])) break;
#pragma unroll
      for (int s = 0; s < 2; ++s) {
        if (go[s]) {
          float sv;
          F3 dummy;
          if (SINGLE) {
            sv = sdf_eval<false, float>(p, fr, as_x3(xo[s] + t[s] * dro[s]), dummy);
          } else {
            sv = __int_as_float(0x7f800000);
            for (int k = 0; k < p.K; ++k) {
              ObjFrameD f2d;
              const ObjFrame f2 = make_frame(p, e, k, RLd, pLd, f2d);
              sv = fminf(sv, sdf_eval<false, float>(p, f2, as_x3(f2.c + mul(f2.M, xj[s] + t[s] * nj[s])), dummy));
            }
          }
          const float tn = fminf(t[s] + fmaxf(sv, 0.f), p.r_prox);
          go[s] = (tn != t[s]) && (tn < p.r_prox);
          t[s] = tn;
        }
      }
    }
    float pr[2];
#pragma unroll
    for (int s = 0; s < 2; ++s) pr[s] = (act[s] && p.march_steps >= 0) ? p.r_prox - t[s] : 0.f;
    if (vec_ok) __stcs(reinterpret_cast<float2*>(p.prox + j0), make_float2(pr[0], pr[1]));
    else {
#pragma unroll
      for (int s = 0; s < 2; ++s)
        if (valid[s]) st_stream(p.prox + j0 + s, pr[s]);
    }
  }
}

// ---------------------------------------------------------------------------------------
// Bank re-tiling: linear [G,N,N,N] (x fastest) -> quad layout (see header comment).
// ---------------------------------------------------------------------------------------
__global__ void ts_retile_kernel(const float* __restrict__ src, float4* __restrict__ dst, int G, int N) {
  const size_t per = (size_t)(N - 1) * (N - 1) * N;
  const size_t total = per * G;
  for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
    const size_t g = idx / per;
    size_t r = idx - g * per;
    const int k = (int)(r % N);
    r /= N;
    const int i = (int)(r % (N - 1)), j = (int)(r / (N - 1));
    const float* s = src + g * (size_t)N * N * N + ((size_t)k * N + j) * N + i;
    dst[idx] = make_float4(s[0], s[1], s[N], s[N + 1]);
  }
}

__global__ void ts_reset_counters_kernel(uint32_t* reset_step, uint32_t* episode, const uint8_t* mask, int E,
                                         uint32_t gstep) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= E) return;
  if (mask && !mask[e]) return;
  reset_step[e] = gstep;
  episode[e] += 1;
}

// Zeroes the state of the masked envs and re-draws their dead flags (Eq. 28, D5): Philox
// stream 2 at n = 0, dead iff word0 < floor(p_dead 2^32).  One thread per (env, patch, lane).
__global__ void ts_reset_state_kernel(const __grid_constant__ TsStepParams p, const uint8_t* mask, uint32_t thr, int nh) {
  const long long gt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long gw = gt >> 5;
  const int lane = (int)(gt & 31);
  if (gw >= (long long)p.E * p.P) return;
  const int e = (int)(gw / p.P), pi = (int)(gw - (long long)e * p.P);
  if (mask && !mask[e]) return;
  const TsPatch pt = p.patches[pi];
  const size_t blk = (size_t)e * p.P + pi;
  const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
  if (p.st_hyst)
    for (int r = 0; r < nh; ++r) p.st_hyst[blk * (nh * 32) + r * 32 + lane] = z4;
  if (p.st_drift)
    for (int r = 0; r < 3; ++r) p.st_drift[blk * (3 * 32) + r * 32 + lane] = z4;
  const uint32_t ep4 = p.episode[e] << 4;
  for (int s = 0; s < 2; ++s) {
    const int i = 2 * lane + s;
    if (i >= pt.n) continue;
    const int t = pt.start + i;
    uint8_t fl = 0;
    if (p.noise_enable && pt.link >= 0 && p.tx_pos[t].w > 0.f) {
      const uint4 w = philox4x32_10(make_uint4(p.env_id_base + (uint32_t)e, (uint32_t)t, 0u, ep4 | 2u), p.seed_lo, p.seed_hi);
      fl = (w.x < thr) ? 2 : 0;
    }
    p.st_flags[(size_t)e * p.T + t] = fl;
  }
}

}  // namespace

unsigned long long ts_bank_elems_per_grid(int N) { return (unsigned long long)(N - 1) * (N - 1) * N; }

int ts_launch_step(const TsStepParams& p, void* stream) {
  const long long warps = (long long)p.E * p.P;
  const long long blocks = (warps * 32 + TS_BLOCK - 1) / TS_BLOCK;
  if (blocks <= 0 || blocks > 0x7fffffffLL) return (int)cudaErrorInvalidConfiguration;
  if (p.K == 1)
    ts_step_kernel<true><<<(unsigned)blocks, TS_BLOCK, 0, (cudaStream_t)stream>>>(p);
  else
    ts_step_kernel<false><<<(unsigned)blocks, TS_BLOCK, 0, (cudaStream_t)stream>>>(p);
  return (int)cudaGetLastError();
}

int ts_launch_retile(const float* src, float4* dst, int G, int N, void* stream) {
  if (G <= 0) return 0;
  ts_retile_kernel<<<148 * 8, 256, 0, (cudaStream_t)stream>>>(src, dst, G, N);
  return (int)cudaGetLastError();
}

int ts_launch_reset_counters(uint32_t* reset_step, uint32_t* episode, const uint8_t* mask, int E, uint32_t gstep,
                             void* stream) {
  ts_reset_counters_kernel<<<(E + 255) / 256, 256, 0, (cudaStream_t)stream>>>(reset_step, episode, mask, E, gstep);
  return (int)cudaGetLastError();
}

int ts_launch_reset_state(const TsStepParams& p, const uint8_t* mask, uint32_t thr, int nh, void* stream) {
  const long long threads = (long long)p.E * p.P * 32;
  const long long blocks = (threads + 255) / 256;
  ts_reset_state_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(p, mask, thr, nh);
  return (int)cudaGetLastError();
}
