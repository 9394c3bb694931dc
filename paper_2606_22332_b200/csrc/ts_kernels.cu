// Hand-written sm_100a kernels of the batched tactile readout.  Citations: "P:NNN" = line of
// the paper text (App. A = P:172-359); "D*/Q*/O*" = readings listed in DESIGN.md.
//
// Mapping: ONE THREAD PER (environment, taxel slot); a block owns one "patch group" of one
// environment: up to TS_BLOCK consecutive taxel slots made of whole patches (packed on the
// host, ts_api.cu).  Per block:
//   phase 0  (own launch, ts_frames_kernel) one thread per (env, patch link, object) builds the relative pose in
//            DOUBLE into frames_g; the step kernel's block fetches its span with one TMA bulk copy on an mbarrier;
//   phase 1  per taxel: x_o = c + M x_j (double), phi (double), depth, Schmitt contact bit;
//   phase 2  proximity march along a_j (fp32; evaluation 0 is the phase-1 query);
//   phase 3  kinematic force/torque in double for warps that touch anything, rounded once;
//   phase 4  noise chain: hysteresis -> crosstalk (neighbours through shared memory) ->
//            Philox/Box-Muller random-walk drift -> dead taxels;
//   phase 5  elastomer marker dilation per patch warp as FP64 tensor-core products (DMMA.8x8x4) of the separable tables.
// Outputs go straight from registers to global memory with streaming stores; shared memory is kept
// at 10 KB per block because it comes out of the L1 that serves the SDF gathers.
//
// Why double in phases 0/1/3/5: outputs are compared element by
// element at rtol 1e-4 / atol 1e-6.  d = R - phi feeds f ~ d^1.2, the marker sum multiplies
// h = -phi by s_d = 100 over up to 64 sources, and a small component of a 3 N force needs the
// contact normal to ~1e-7.  fp32 positions (ulp 4e-9 m at 5 cm) give neither.  B200 issues DFMA
// at half the FFMA rate; the double chain is ~250 instructions per touching taxel.
//
// Bank layout ("quad"): for every grid, Q[(j*(N-1) + i)*N + k] = float4(phi(i,j,k), phi(i+1,j,k),
// phi(i,j+1,k), phi(i+1,j+1,k)), i,j in [0,N-2], k in [0,N-1].  The 8 corners of cell (i,j,k) are
// the two consecutive float4 Q[..k], Q[..k+1]: one 32-byte span, two LDG.128 instead of eight
// scattered LDG.32 (the L1 wavefront count of the gather is what bounds the SDF path).
#include <cuda_runtime.h>

#include <cstdint>
#include <mutex>

#include "ts_internal.h"

#ifndef TS_MARCH_LATE
#define TS_MARCH_LATE 0  // 1: proximity march after the noise chain (experiment)
#endif
#ifndef TS_PDL
#define TS_PDL 2  // 1: step kernel launched as a programmatic dependent of ts_frames_kernel (griddepcontrol);
                  // 2: also the NEXT step's frames kernel as a dependent of this step kernel (see ts_launch_frames)
#endif

namespace {

__device__ __forceinline__ unsigned long long globaltimer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}

struct F3 {
  float x, y, z;
};
struct D3 {
  double x, y, z;
};
__device__ __forceinline__ F3 mk3(float x, float y, float z) { return F3{x, y, z}; }
__device__ __forceinline__ F3 operator+(F3 a, F3 b) { return F3{a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ F3 operator*(float s, F3 a) { return F3{s * a.x, s * a.y, s * a.z}; }
__device__ __forceinline__ float dot(F3 a, F3 b) { return fmaf(a.x, b.x, fmaf(a.y, b.y, a.z * b.z)); }

__device__ __forceinline__ D3 operator+(D3 a, D3 b) { return D3{a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ D3 operator-(D3 a, D3 b) { return D3{a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ D3 operator*(double s, D3 a) { return D3{s * a.x, s * a.y, s * a.z}; }
__device__ __forceinline__ double dot(D3 a, D3 b) { return fma(a.x, b.x, fma(a.y, b.y, a.z * b.z)); }
__device__ __forceinline__ D3 cross(D3 a, D3 b) {
  return D3{fma(a.y, b.z, -a.z * b.y), fma(a.z, b.x, -a.x * b.z), fma(a.x, b.y, -a.y * b.x)};
}
__device__ __forceinline__ D3 ld3d(const float* p) { return D3{(double)__ldg(p), (double)__ldg(p + 1), (double)__ldg(p + 2)}; }
__device__ __forceinline__ D3 ldv(const double* p) { return D3{p[0], p[1], p[2]}; }
// y = R v, y = R^T v for a row-major 3x3 of doubles
__device__ __forceinline__ D3 mulR(const double* R, D3 v) {
  return D3{fma(R[0], v.x, fma(R[1], v.y, R[2] * v.z)), fma(R[3], v.x, fma(R[4], v.y, R[5] * v.z)),
            fma(R[6], v.x, fma(R[7], v.y, R[8] * v.z))};
}
__device__ __forceinline__ D3 mulRT(const double* R, D3 v) {
  return D3{fma(R[0], v.x, fma(R[3], v.y, R[6] * v.z)), fma(R[1], v.x, fma(R[4], v.y, R[7] * v.z)),
            fma(R[2], v.x, fma(R[5], v.y, R[8] * v.z))};
}

// sqrt / reciprocal sqrt of a double to ~1e-13 relative: MUFU.RSQ seed + one Newton step in
// double (a correctly rounded DSQRT costs ~4x more and its last bits are not needed).
__device__ __forceinline__ double dsqrt_n(double s) {
  const float sf = (float)s;
  if (!(sf > 0.f)) return 0.0;
  const float rs = rsqrtf(sf);
  const double r0 = (double)(sf * rs);
  const double e = fma(-r0, r0, s);
  return fma(e, (double)(0.5f * rs), r0);
}
__device__ __forceinline__ double drsqrt_n(double s) {  // s > 0
  const double y0 = (double)rsqrtf((float)s);
  const double e = fma(-s * y0, y0, 1.0);
  return fma(0.5 * y0, e, y0);
}

// O0: rotation of a quaternion (w,x,y,z), used as given.
__device__ __forceinline__ void quat_Rd(const float* q4, double* R) {
  const float4 q = __ldg(reinterpret_cast<const float4*>(q4));
  const double w = q.x, x = q.y, y = q.z, z = q.w;
  R[0] = 1.0 - 2.0 * (y * y + z * z); R[1] = 2.0 * (x * y - w * z);       R[2] = 2.0 * (x * z + w * y);
  R[3] = 2.0 * (x * y + w * z);       R[4] = 1.0 - 2.0 * (x * x + z * z); R[5] = 2.0 * (y * z - w * x);
  R[6] = 2.0 * (x * z - w * y);       R[7] = 2.0 * (y * z + w * x);       R[8] = 1.0 - 2.0 * (x * x + y * y);
}

// Relative pose of (sensor link of a patch, object k), in shared memory.  x_o = c + M x_j maps
// link-frame points to the object frame; p_L - p_O is formed BEFORE rotating.
struct FrameS {
  double M[9];     // R_O^T R_L
  double c[3];     // R_O^T (p_L - p_O)
  double wO[3];    // R_L^T w_O   (link-frame velocity terms of Eq. 4-6)
  double wL[3];    // R_L^T w_L
  double vbar[3];  // R_L^T (v_O - v_L)
  double cbar[3];  // R_L^T (p_L - p_O)
  float prm[4];
  int type;
  float dirf[3];   // M n: march direction of the patch normal in the object frame (fp32)
};                 // 224 bytes: a multiple of 16 (the step kernel's bulk copy moves whole records)
static_assert(sizeof(FrameS) == 224, "FrameS layout");

// One frame is built by SEVEN threads so that the dependent double-precision chain the whole block
// waits for stays short (~60 instructions): "row" items r = 0..2 (row r of M and c[r]) run in the lower
// half of the block, "vector" items s = 0..3 (wO, wL, vbar, cbar) in the upper half, so a warp never
// executes both code paths.
__device__ __forceinline__ void build_frame_row(const TsStepParams& p, int e, int link, int pidx, int k, int r, FrameS& F) {
  if (link < 0) return;
  const float4 na = __ldg(&p.patches[pidx].na);
  const size_t ek = (size_t)e * p.K + k, el = (size_t)e * p.L + link;
  double RL[9];
  quat_Rd(p.link_quat + el * 4, RL);
  const D3 d = ld3d(p.link_pos + el * 3) - ld3d(p.obj_pos + ek * 3);
  // column r of R_O, with (i, j, k) = (r, r+1, r+2) mod 3: R[i][i] = 1 - 2(q_j^2 + q_k^2),
  // R[j][i] = 2(q_i q_j + w q_k), R[k][i] = 2(q_i q_k - w q_j)
  const float4 q = __ldg(reinterpret_cast<const float4*>(p.obj_quat + ek * 4));
  const double w = q.x;
  const double qi = r == 0 ? q.y : (r == 1 ? q.z : q.w);
  const double qj = r == 0 ? q.z : (r == 1 ? q.w : q.y);
  const double qk = r == 0 ? q.w : (r == 1 ? q.y : q.z);
  const double ci = 1.0 - 2.0 * (qj * qj + qk * qk), cj = 2.0 * (qi * qj + w * qk), ck = 2.0 * (qi * qk - w * qj);
  // rows of R_O's column r in canonical order (row 0, 1, 2)
  const double o0 = r == 0 ? ci : (r == 1 ? ck : cj);
  const double o1 = r == 0 ? cj : (r == 1 ? ci : ck);
  const double o2 = r == 0 ? ck : (r == 1 ? cj : ci);
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const double m = fma(o0, RL[c], fma(o1, RL[3 + c], o2 * RL[6 + c]));
    F.M[r * 3 + c] = m;
  }
  const double cr = fma(o0, d.x, fma(o1, d.y, o2 * d.z));
  F.c[r] = cr;
  F.dirf[r] = (float)fma(F.M[r * 3], (double)na.x, fma(F.M[r * 3 + 1], (double)na.y, F.M[r * 3 + 2] * (double)na.z));
}

__device__ __forceinline__ void build_frame_vec(const TsStepParams& p, int e, int link, int k, int sub, FrameS& F) {
  const size_t ek = (size_t)e * p.K + k;
  if (sub == 3) {
    F.type = (link >= 0) ? __ldg(p.g_type + ek) : TS_GEOM_NONE;
    const float4 prm = __ldg(p.g_params + ek);
    F.prm[0] = prm.x; F.prm[1] = prm.y; F.prm[2] = prm.z; F.prm[3] = prm.w;
  }
  if (link < 0) return;
  const size_t el = (size_t)e * p.L + link;
  double RL[9];
  quat_Rd(p.link_quat + el * 4, RL);
  // sub 0: w_O, 1: w_L, 2: v_O - v_L, 3: p_L - p_O; all rotated into the link frame by R_L^T
  const float* a = sub == 0 ? p.obj_angvel + ek * 3 : (sub == 1 ? p.link_angvel + el * 3 : (sub == 2 ? p.obj_linvel + ek * 3 : p.link_pos + el * 3));
  const float* b = sub == 2 ? p.link_linvel + el * 3 : p.obj_pos + ek * 3;
  D3 v = ld3d(a);
  if (sub >= 2) v = v - ld3d(b);
  const D3 o = mulRT(RL, v);
  double* dst = F.wO + 3 * sub;  // wO, wL, vbar, cbar are consecutive
  dst[0] = o.x; dst[1] = o.y; dst[2] = o.z;
}

// Phase 0 as its own launch: one thread per (env, patch, object) builds the whole frame and writes it to frames_g (block
// order of the step kernel).  Inside the step kernel the same arithmetic sat in front of a block barrier and took
// ~19 % of every block's lifetime (a ~250-instruction dependent double-precision chain behind a DRAM round trip, with
// 6 of 8 warps waiting); here it is 410 k independent threads, and the step kernel's blocks receive their frames with
// one TMA bulk copy.
__global__ void __launch_bounds__(128) ts_frames_kernel(const __grid_constant__ TsStepParams p) {
  // Each warp stages its 32 consecutive frames in shared memory and writes them out as one contiguous, fully coalesced
  // run: per-thread rows straight to global memory cost 32 sectors per store request (ncu: lg_throttle 4.2 per issue,
  // 47 us).  The fields go straight into the thread's staging row (no register image of the record: 96 -> ~56
  // registers); the row stride of 232 bytes (= 58 words) spreads the 16 lanes of an 8-byte store over distinct banks.
  constexpr int STRIDE = (int)sizeof(FrameS) + 8;
  __shared__ __align__(16) unsigned char stage[128 * STRIDE];
#if TS_PDL
  asm volatile("griddepcontrol.launch_dependents;");   // once every block of this grid is resident, the step kernel's may start
#endif
#if TS_PDL >= 2
  // Launched as a programmatic dependent (ts_launch_frames): the blocks may become resident while the kernel in front of
  // this one in the stream is in its last wave; they wait here until it -- the previous step kernel, or whatever the
  // caller enqueued to produce this step's poses -- has completed and its writes are visible.  (Reading the poses before
  // this wait, which is legal only for inputs that are older than the previous step, measured no faster.)
  asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
  if (p.clock && threadIdx.x == 0) atomicMin(p.clock, globaltimer_ns());   // device-side clock: first block's start of work
  const int PK = p.P * p.K;
  const long long total = (long long)p.E * PK;
  const long long gt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  FrameS& F = *reinterpret_cast<FrameS*>(stage + (size_t)threadIdx.x * STRIDE);
  int link = -1;
  if (gt < total) {
    // frames are stored in BLOCK order of the step kernel (row bx = frames of env env_perm[bx]), so that a block's bulk
    // copy needs no env lookup in front of it and the rows of the blocks scheduled next sit at a fixed distance ahead
    const int bx = (int)(gt / PK), f = (int)(gt - (long long)bx * PK);
    const int e = p.env_perm ? __ldg(p.env_perm + bx) : bx;
    const int pidx = f / p.K, k = f - pidx * p.K;
    link = __ldg(p.patch_link + pidx);
    if (link < 0) {   // filtered link: everything but type / prm stays zero
#pragma unroll
      for (int i = 0; i < (int)(sizeof(FrameS) / 8); ++i) reinterpret_cast<uint2*>(&F)[i] = make_uint2(0u, 0u);
    }
#pragma unroll
    for (int r = 0; r < 3; ++r) build_frame_row(p, e, link, pidx, k, r, F);
#pragma unroll
    for (int sub = 0; sub < 4; ++sub) build_frame_vec(p, e, link, k, sub, F);
  }
  __syncwarp();
  const int lane = threadIdx.x & 31, w0 = threadIdx.x & ~31;
  const long long g0 = (long long)blockIdx.x * blockDim.x + w0;              // first frame of this warp
  constexpr int W8 = (int)(sizeof(FrameS) / 8);                              // 8-byte words per record
  const int n8 = (int)(total - g0 < 32 ? (total - g0 > 0 ? total - g0 : 0) : 32) * W8;
  const unsigned char* wsrc = stage + (size_t)w0 * STRIDE;
  uint2* wdst = reinterpret_cast<uint2*>(reinterpret_cast<FrameS*>(p.frames_g) + g0);
#pragma unroll
  for (int i = 0; i < W8; ++i) {
    const int q = i * 32 + lane, fr = q / W8, part = q - fr * W8;
    if (q < n8) wdst[q] = *reinterpret_cast<const uint2*>(wsrc + fr * STRIDE + part * 8);
  }
}

// ---------------------------------------------------------------------------------------
// O2 in double: signed distance and (unnormalised, object-frame) gradient of one geometry at
// the object-frame point x.  Used once per taxel (the first query).
// ---------------------------------------------------------------------------------------
struct CellD {  // trilinear cell around x: corners, in-cell fractions, outside-grid offset (voxels)
  float4 A, B;  // (c000,c100,c010,c110), (c001,c101,c011,c111)
  double fx, fy, fz;
  double ox, oy, oz;
  bool outside;
};

__device__ __forceinline__ void clamp01(double& f, double& o, bool& outside) {
  const float ff = (float)f;
  o = 0.0;
  if (ff < 0.f || ff > 1.f) {  // outside the grid on this axis (O2 extension); rare
    const double c = ff < 0.f ? 0.0 : 1.0;
    o = f - c;
    f = c;
    outside = true;
  }
}

__device__ __forceinline__ void grid_cell_d(const TsStepParams& p, int gid, D3 x, CellD& C) {
  const int N = p.grid_n;
  const double half = 0.5 * (double)(N - 1);
  const double ux = fma(x.x, p.inv_voxel_d, half), uy = fma(x.y, p.inv_voxel_d, half), uz = fma(x.z, p.inv_voxel_d, half);
  // cell index from the fp32 image of u: a one-ulp slip across a face only moves the (continuous)
  // interpolant by ~1e-11 m and lands in the comparator's voxel-face band for the gradient.
  const int i0 = min(max(__float2int_rd((float)ux), 0), N - 2);
  const int j0 = min(max(__float2int_rd((float)uy), 0), N - 2);
  const int k0 = min(max(__float2int_rd((float)uz), 0), N - 2);
  C.fx = ux - (double)i0; C.fy = uy - (double)j0; C.fz = uz - (double)k0;
  C.outside = false;
  clamp01(C.fx, C.ox, C.outside);
  clamp01(C.fy, C.oy, C.outside);
  clamp01(C.fz, C.oz, C.outside);
  const float4* q = p.bank + (size_t)gid * p.grid_stride + ((size_t)(j0 * (N - 1) + i0) * N + k0);
  C.A = __ldg(q);
  C.B = __ldg(q + 1);
}

__device__ __forceinline__ double grid_value_d(const TsStepParams& p, const CellD& C) {
  const double c000 = C.A.x, c100 = C.A.y, c010 = C.A.z, c110 = C.A.w;
  const double c001 = C.B.x, c101 = C.B.y, c011 = C.B.z, c111 = C.B.w;
  const double a0 = fma(C.fx, c100 - c000, c000), a1 = fma(C.fx, c110 - c010, c010);
  const double b0 = fma(C.fx, c101 - c001, c001), b1 = fma(C.fx, c111 - c011, c011);
  const double lo = fma(C.fy, a1 - a0, a0), hi = fma(C.fy, b1 - b0, b0);
  double phi = fma(C.fz, hi - lo, lo);
  if (C.outside) phi += (double)p.voxel * dsqrt_n(fma(C.ox, C.ox, fma(C.oy, C.oy, C.oz * C.oz)));
  return phi;
}

// exact derivative of the trilinear interpolant in the cell; the common factor 1/h_v is dropped
__device__ __forceinline__ D3 grid_grad_d(const CellD& C) {
  const double c000 = C.A.x, c100 = C.A.y, c010 = C.A.z, c110 = C.A.w;
  const double c001 = C.B.x, c101 = C.B.y, c011 = C.B.z, c111 = C.B.w;
  const double a0 = fma(C.fx, c100 - c000, c000), a1 = fma(C.fx, c110 - c010, c010);
  const double b0 = fma(C.fx, c101 - c001, c001), b1 = fma(C.fx, c111 - c011, c011);
  const double lo = fma(C.fy, a1 - a0, a0), hi = fma(C.fy, b1 - b0, b0);
  const double gy0 = 1.0 - C.fy, gz0 = 1.0 - C.fz;
  const double dxa = fma(C.fy, c110 - c010, gy0 * (c100 - c000)), dxb = fma(C.fy, c111 - c011, gy0 * (c101 - c001));
  return D3{fma(C.fz, dxb, gz0 * dxa), fma(C.fz, b1 - b0, gz0 * (a1 - a0)), hi - lo};
}

__device__ __forceinline__ double phi_d(const TsStepParams& p, int type, const float* prm, D3 x) {
  switch (type) {
    case TS_GEOM_SPHERE:
      return dsqrt_n(dot(x, x)) - (double)prm[0];
    case TS_GEOM_BOX: {
      const double wx = fabs(x.x) - (double)prm[0], wy = fabs(x.y) - (double)prm[1], wz = fabs(x.z) - (double)prm[2];
      const double px = fmax(wx, 0.0), py = fmax(wy, 0.0), pz = fmax(wz, 0.0);
      return dsqrt_n(fma(px, px, fma(py, py, pz * pz))) + fmin(fmax(wx, fmax(wy, wz)), 0.0);
    }
    case TS_GEOM_CAPSULE: {
      const double h = (double)prm[1];
      const double zc = fmin(fmax(x.z, -h), h);
      const D3 y = D3{x.x, x.y, x.z - zc};
      return dsqrt_n(dot(y, y)) - (double)prm[0];
    }
    case TS_GEOM_SDF: {
      CellD C;
      grid_cell_d(p, (int)prm[0], x, C);
      return grid_value_d(p, C);
    }
    default:
      return __longlong_as_double(0x7ff0000000000000LL);
  }
}

// unnormalised gradient; the zero vector flags a singular point (Q2/Q7 handled by the caller)
__device__ __forceinline__ D3 grad_d(const TsStepParams& p, int type, const float* prm, D3 x) {
  switch (type) {
    case TS_GEOM_SPHERE:
      return dot(x, x) < 1e-24 ? D3{0.0, 0.0, 1.0} : x;
    case TS_GEOM_BOX: {
      const double wx = fabs(x.x) - (double)prm[0], wy = fabs(x.y) - (double)prm[1], wz = fabs(x.z) - (double)prm[2];
      const double sx = x.x < 0.0 ? -1.0 : 1.0, sy = x.y < 0.0 ? -1.0 : 1.0, sz = x.z < 0.0 ? -1.0 : 1.0;
      if (fmax(wx, fmax(wy, wz)) > 0.0) return D3{sx * fmax(wx, 0.0), sy * fmax(wy, 0.0), sz * fmax(wz, 0.0)};
      if (wx >= wy && wx >= wz) return D3{sx, 0.0, 0.0};  // interior: axis of the largest w, ties -> lowest index (Q7)
      if (wy >= wz) return D3{0.0, sy, 0.0};
      return D3{0.0, 0.0, sz};
    }
    case TS_GEOM_CAPSULE: {
      const double h = (double)prm[1];
      const double zc = fmin(fmax(x.z, -h), h);
      const D3 y = D3{x.x, x.y, x.z - zc};
      return dot(y, y) < 1e-24 ? D3{0.0, 0.0, 1.0} : y;
    }
    case TS_GEOM_SDF: {
      CellD C;
      grid_cell_d(p, (int)prm[0], x, C);
      return grid_grad_d(C);
    }
    default:
      return D3{0.0, 0.0, 0.0};
  }
}

// ---------------------------------------------------------------------------------------
// O2 in fp32, value only: the march evaluations (prox tolerance 1e-6 m; fp32 gives ~1e-8).
// ---------------------------------------------------------------------------------------
// Packed fp32 pairs (Blackwell FADD2 / FFMA2: one issue slot for two lanes of arithmetic; a scalar operand is broadcast).
__device__ __forceinline__ unsigned long long pk2(float2 a) { unsigned long long r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a.x), "f"(a.y)); return r; }
__device__ __forceinline__ float2 upk2(unsigned long long a) { float2 r; asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(a)); return r; }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { unsigned long long d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(pk2(a)), "l"(pk2(b))); return upk2(d); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { unsigned long long d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(pk2(a)), "l"(pk2(b)), "l"(pk2(c))); return upk2(d); }
__device__ __forceinline__ float2 bc2(float a) { return make_float2(a, a); }

// A = (c000, c100, c010, c110), B = (c001, c101, c011, c111): blend along y and z on (x = 0, x = 1) pairs, then along x
// (8 instructions instead of 14; the blend order only changes the rounding, ~1e-9 m against the 1e-6 m prox tolerance).
__device__ __forceinline__ float trilerp(float4 A, float4 B, float fx, float fy, float fz) {
  const float2 a0 = make_float2(A.x, A.y), a1 = make_float2(A.z, A.w), b0 = make_float2(B.x, B.y), b1 = make_float2(B.z, B.w);
  const float2 a = fma2(bc2(fy), sub2(a1, a0), a0);
  const float2 b = fma2(bc2(fy), sub2(b1, b0), b0);
  const float2 c = fma2(bc2(fz), sub2(b, a), a);
  return fmaf(fx, c.y - c.x, c.x);
}

// general point (clamps + outside-grid extension); u = voxel coordinates
__device__ __forceinline__ float grid_value_f(const TsStepParams& p, const float4* bank_g, F3 u) {
  const int N = p.grid_n;
  const float top = (float)(N - 1);
  const float cx = fminf(fmaxf(u.x, 0.f), top), cy = fminf(fmaxf(u.y, 0.f), top), cz = fminf(fmaxf(u.z, 0.f), top);
  const int i0 = min((int)cx, N - 2), j0 = min((int)cy, N - 2), k0 = min((int)cz, N - 2);
  const float4* q = bank_g + ((size_t)(j0 * (N - 1) + i0) * N + k0);
  float phi = trilerp(__ldg(q), __ldg(q + 1), cx - (float)i0, cy - (float)j0, cz - (float)k0);
  const float ox = u.x - cx, oy = u.y - cy, oz = u.z - cz;
  const float o2 = fmaf(ox, ox, fmaf(oy, oy, oz * oz));
  if (o2 > 0.f) phi += p.voxel * sqrtf(o2);
  return phi;
}

// MUFU.SQRT (relative error <= 2^-22): |x| <= 0.1 m gives <= 3e-8 m per march evaluation, <= 5e-7 m over
// 16 evaluations in the worst case against the 1e-6 m prox tolerance; the IEEE sqrtf costs 8 instructions.
__device__ __forceinline__ float sqrt_approx(float x) {
  float r;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

__device__ __forceinline__ float prim_value_f(int type, const float* prm, F3 x) {
  switch (type) {
    case TS_GEOM_SPHERE:
      return sqrt_approx(dot(x, x)) - prm[0];
    case TS_GEOM_BOX: {
      const float wx = fabsf(x.x) - prm[0], wy = fabsf(x.y) - prm[1], wz = fabsf(x.z) - prm[2];
      const float px = fmaxf(wx, 0.f), py = fmaxf(wy, 0.f), pz = fmaxf(wz, 0.f);
      return sqrt_approx(fmaf(px, px, fmaf(py, py, pz * pz))) + fminf(fmaxf(wx, fmaxf(wy, wz)), 0.f);
    }
    case TS_GEOM_CAPSULE: {
      const float zc = fminf(fmaxf(x.z, -prm[1]), prm[1]);
      const F3 y = mk3(x.x, x.y, x.z - zc);
      return sqrt_approx(dot(y, y)) - prm[0];
    }
    default:
      return __int_as_float(0x7f800000);
  }
}

__device__ __forceinline__ float phi_f(const TsStepParams& p, int type, const float* prm, F3 x) {
  if (type == TS_GEOM_SDF) {
    const float half = 0.5f * (float)(p.grid_n - 1);
    const F3 u = mk3(fmaf(x.x, p.inv_voxel, half), fmaf(x.y, p.inv_voxel, half), fmaf(x.z, p.inv_voxel, half));
    return grid_value_f(p, p.bank + (size_t)(int)prm[0] * p.grid_stride, u);
  }
  return prim_value_f(type, prm, x);
}

// ---------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al. 2011), counter = (env, taxel, n, episode<<4 | stream) (O8).
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c.x, p1 = (uint64_t)0xCD9E8D57u * c.z;
    c = make_uint4((uint32_t)(p1 >> 32) ^ c.y ^ k0, (uint32_t)p1, (uint32_t)(p0 >> 32) ^ c.w ^ k1, (uint32_t)p0);
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  return c;
}

// Box-Muller on a word pair (O8): u = (2 (w >> 9) + 1) 2^-24 (exact in fp32, never 0 or 1),
// z0 = sqrt(-2 ln u_a) cos(2 pi u_b), z1 = ... sin(...).
//  * -2 ln u_a: MUFU.LG2 has an ABSOLUTE error of ~2^-22 near u = 1, so for 1 - u < 1/64 the
//    series of -ln(1 - v) (v = 1 - u is exact) is used instead; relative error of L <= ~1e-5.
//  * the angle is reduced EXACTLY in integers to [-pi, pi) (k_b is a 24-bit integer), then MUFU.SIN/COS
//    (abs error ~4e-7 there).
// Error of z <= ~1e-5 |z| + 4e-7 r, i.e. < 1e-8 N per step at sigma = 1e-3 N (tolerance 1e-6).
__device__ __forceinline__ float lg2_ftz(float x) {  // MUFU.LG2 without the denormal fix-up of __log2f (x >= 2^-24 here)
  float r;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float rsqrt_ftz(float x) {  // MUFU.RSQ without the denormal fix-up of rsqrtf (x >= 1e-7 here)
  float r;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ void box_muller(uint32_t wa, uint32_t wb, float& z0, float& z1) {
  const float ua = (float)(2u * (wa >> 9) + 1u) * 5.9604644775390625e-8f;
  const float v = 1.f - ua;  // exact
  const float Ls = 2.f * v * fmaf(v, fmaf(v, fmaf(v, 0.25f, 0.33333334f), 0.5f), 1.f);  // -2 ln(1-v), v < 1/64: rel 2e-9
  const float Ll = -1.3862943611198906f * lg2_ftz(ua);                                  // -2 ln 2 * log2 u
  const float L = (v < 0.015625f) ? Ls : Ll;                                           // L >= -2 ln(1 - 2^-24) = 1.2e-7
  const float r = L * rsqrt_ftz(L);
  // angle 2 pi k_b / 2^24 mapped to [-pi, pi) by sign-extending the 24-bit integer (same sin / cos);
  // MUFU.SIN / MUFU.COS have an absolute error of ~4e-7 on that range
  const int kb = ((int)((2u * (wb >> 9) + 1u) << 8)) >> 8;
  const float th = (float)kb * 3.7450703e-7f;  // 2 pi / 2^24
  z0 = r * __cosf(th);
  z1 = r * __sinf(th);
}

// six channels of one taxel ([E,T,6] row, 24 bytes, 8-byte aligned): three streaming 8-byte stores
__device__ __forceinline__ void store6(float* dst, const float* v) {
  float2* d2 = reinterpret_cast<float2*>(dst);
  __stcs(d2, make_float2(v[0], v[1]));
  __stcs(d2 + 1, make_float2(v[2], v[3]));
  __stcs(d2 + 2, make_float2(v[4], v[5]));
}

// D (8 x 8) += A (8 x 4, row) B (4 x 8, col) on the FP64 tensor cores: lane = 4 g + m holds A[g][m], B[m][g], D[g][2m], D[g][2m+1].
__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// ---- TMA bulk copy global -> shared memory, completion on an mbarrier (cp.async.bulk, SASS UBLKCP) -------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, unsigned bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@!p bra WAIT_%=;\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

#define TS_FULL 0xffffffffu
#ifndef TS_HYST_STORE_LATE
#define TS_HYST_STORE_LATE 1
#endif
#ifndef TS_PF_AHEAD
#define TS_PF_AHEAD 1184  // blocks: ~1.3 waves of 6 resident blocks x 148 SMs
#endif
#ifndef TS_GRID_GFAST
#define TS_GRID_GFAST 1  // launch order: the patch groups of one env are adjacent (its frames, state and output rows are touched together)
#endif
#ifndef TS_MIN_BLOCKS
#define TS_MIN_BLOCKS 5
#endif

// ---------------------------------------------------------------------------------------
// The fused step kernel: S1-S8 of DESIGN.md; block = (env, patch group), thread = taxel slot.
// ---------------------------------------------------------------------------------------
// ---------------------------------------------------------------------------------------
// S8: noise chain of one taxel (O8): hysteresis -> crosstalk -> drift -> dead.  Shared by the fused
// step kernel and the stand-alone noise kernel.
// ---------------------------------------------------------------------------------------
// Streaming float2 load that does not allocate in L1 (the state is read exactly once; L1 is kept for the
// SDF gathers and the layout tables).
__device__ __forceinline__ float2 ld_stream2(const float2* p) {
  float2 v;
  asm volatile("ld.global.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p) : "memory");
  return v;
}

struct NoiseState {
  float sY[6], sX[6], sD[6];  // hysteresis y (asym) or xi (maxwell), maxwell x_prev, drift D
};

// HM = hysteresis mode (TS_HYST_*) | 4 if the remaining A.8 knobs (Eq. 25 bias / white noise / quantisation,
// Eq. 27 gain, Eq. 28 stuck value) are on: compile-time, so unused state rows and knobs cost nothing.
template <int HM>
__device__ __forceinline__ void noise_load(const TsStepParams& p, int e, int j, bool valid, NoiseState& ns) {
  constexpr int MODE = HM & 3;
  // 32-bit element indices (ts_create guarantees E * 12 * Tp < 2^32): one IMAD + LEA pair per access
  // instead of 64-bit address arithmetic that the register allocator keeps rematerialising.
  // State rows hold channel PAIRS (float2): [E][nh/2][Tp] and [E][3][Tp], so a warp moves 256 contiguous
  // bytes per access and a taxel needs 3 + 3 loads instead of 6 + 6.
  const unsigned Tp = (unsigned)p.Tp;
  const unsigned ih = (unsigned)e * (MODE == TS_HYST_MAXWELL ? 6u : 3u) * Tp + (unsigned)j;
  const unsigned id = (unsigned)e * 3u * Tp + (unsigned)j;
  const float2* st_h = reinterpret_cast<const float2*>(p.st_hyst);
  const float2* st_d = reinterpret_cast<const float2*>(p.st_drift);
#pragma unroll
  for (int c = 0; c < 6; ++c) { ns.sY[c] = 0.f; ns.sX[c] = 0.f; ns.sD[c] = 0.f; }
  if (valid) {
    if (MODE != TS_HYST_OFF) {
#pragma unroll
      for (int c = 0; c < 3; ++c) { const float2 v = ld_stream2(st_h + (ih + c * Tp)); ns.sY[2 * c] = v.x; ns.sY[2 * c + 1] = v.y; }
    }
    if (MODE == TS_HYST_MAXWELL) {
#pragma unroll
      for (int c = 0; c < 3; ++c) { const float2 v = ld_stream2(st_h + (ih + (3 + c) * Tp)); ns.sX[2 * c] = v.x; ns.sX[2 * c + 1] = v.y; }
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) { const float2 v = ld_stream2(st_d + (id + c * Tp)); ns.sD[2 * c] = v.x; ns.sD[2 * c + 1] = v.y; }
  }
}

// The 12 (18) per-taxel state words of the noise chain are only PREFETCHED into L2 early in the kernel (one
// request per 128-byte line of a float2 row, i.e. every 16th thread) and loaded right before the chain:
// holding them in registers across the march cost spills at 48 registers per thread (measured 1.48 ->
// 1.41 ms on config 5), and an L2 hit is short enough for 40 resident warps to cover.
template <int HM>
__device__ __forceinline__ void noise_prefetch(const TsStepParams& p, int e, int j0, int jend, int lane) {
  // One request per 128-byte line of the warp's state rows: lane = 2 * row + half (a warp's 32 slots are 256 bytes of a
  // float2 row); every lane forms ONE address (the earlier form had every 16th lane walk all rows: 18 issue slots).
  constexpr int MODE = HM & 3;
  constexpr int NH = MODE == TS_HYST_MAXWELL ? 6 : (MODE == TS_HYST_ASYM ? 3 : 0);
  const int r = lane >> 1, jj = j0 + (lane & 1) * 16;
  if (r < NH + 3 && jj < jend) {
    const unsigned Tp = (unsigned)p.Tp;
    const float2* row = r < NH ? reinterpret_cast<const float2*>(p.st_hyst) + ((unsigned)e * (unsigned)NH + (unsigned)r) * Tp
                               : reinterpret_cast<const float2*>(p.st_drift) + ((unsigned)e * 3u + (unsigned)(r - NH)) * Tp;
    asm volatile("prefetch.global.L2 [%0];" ::"l"(row + jj));
  }
}

// The same prefetch for the whole block by ONE thread: a bulk L2 prefetch (cp.async.bulk.prefetch.L2, SASS UBLKPF) per
// state row of the block's slots [gstart, gstart + gcount), issued from the uniform datapath next to the frames copy:
// ~3 issue slots per warp on average instead of 24 in every warp.  Start and size are rounded outwards to 16 bytes
// (rows are padded to Tp = 32 k slots, so the span stays inside the env's row).
#ifndef TS_STATE_BULK_PF
#define TS_STATE_BULK_PF 1
#endif
template <int HM>
__device__ __forceinline__ void noise_prefetch_bulk(const TsStepParams& p, int e, int gstart, int gcount) {
  constexpr int MODE = HM & 3;
  constexpr int NH = MODE == TS_HYST_MAXWELL ? 6 : (MODE == TS_HYST_ASYM ? 3 : 0);
  const unsigned Tp = (unsigned)p.Tp;
  const unsigned j0 = (unsigned)gstart & ~1u;
  const unsigned bytes = ((((unsigned)(gstart + gcount) + 1u) & ~1u) - j0) * 8u;
  const float2* h = reinterpret_cast<const float2*>(p.st_hyst) + (size_t)((unsigned)e * (unsigned)NH) * Tp + j0;
  const float2* d = reinterpret_cast<const float2*>(p.st_drift) + (size_t)((unsigned)e * 3u) * Tp + j0;
#pragma unroll
  for (int r = 0; r < NH; ++r) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(h + (size_t)r * Tp), "r"(bytes) : "memory");
#pragma unroll
  for (int r = 0; r < 3; ++r) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(d + (size_t)r * Tp), "r"(bytes) : "memory");
}

// Every thread of the block must call this (it contains one __syncthreads).
template <int HM, bool FAST = false>
__device__ __forceinline__ void noise_chain(const TsStepParams& p, int e, int j, unsigned ej, int tid, int patch0, bool valid,
                                            bool act, bool deadb, int meta, const float* ft, const NoiseState& ns,
                                            float* bufB) {
  constexpr int MODE = HM & 3;
  constexpr bool EXT = (HM & 4) != 0;
  const unsigned Tp = (unsigned)p.Tp;
  const unsigned ih = (unsigned)e * (MODE == TS_HYST_MAXWELL ? 6u : 3u) * Tp + (unsigned)j;
  const unsigned id = (unsigned)e * 3u * Tp + (unsigned)j;
  float2* const st_h = reinterpret_cast<float2*>(p.st_hyst);
  float2* const st_d = reinterpret_cast<float2*>(p.st_drift);
  const uint32_t ep4 = __ldg(p.episode + e) << 4;
  const uint32_t env = p.env_id_base + (uint32_t)e;
  float x[6];  // the signal the chain acts on: gamma_bj ft (Eq. 27, R1/R2), gamma = 1 without EXT
#pragma unroll
  for (int c = 0; c < 6; ++c) x[c] = ft[c];
  if (EXT && act && (p.gain_min != 1.f || p.gain_max != 1.f)) {  // stream 3, n = 0: once per episode, recomputed here
    const uint4 w = philox4x32_10(make_uint4(env, (uint32_t)j, 0u, ep4 | 3u), p.seed_lo, p.seed_hi);
    const float u = (float)(2u * (w.x >> 9) + 1u) * 5.9604644775390625e-8f;
    const float g = fmaf(p.gain_max - p.gain_min, u, p.gain_min);
#pragma unroll
    for (int c = 0; c < 6; ++c) x[c] *= g;
  }
  float h[6];
  if (MODE == TS_HYST_ASYM) {  // D3, Q14
#pragma unroll
    for (int c = 0; c < 6; ++c) {
      const float yp = ns.sY[c];
      const float al = (fabsf(x[c]) > fabsf(yp)) ? p.alpha_load : p.alpha_unload;
      h[c] = act ? fmaf(al, x[c] - yp, yp) : 0.f;
    }
    // the new state (= h) is written back AFTER the exchange barrier below (TS_HYST_STORE_LATE)
    if (!TS_HYST_STORE_LATE && valid) {
#pragma unroll
      for (int c = 0; c < 3; ++c) __stcs(st_h + (ih + c * Tp), make_float2(h[2 * c], h[2 * c + 1]));
    }
  } else if (MODE == TS_HYST_MAXWELL) {  // Eq. 29-30
    float zx[6];
#pragma unroll
    for (int c = 0; c < 6; ++c) {
      zx[c] = act ? fmaf(p.decay, ns.sY[c], x[c] - ns.sX[c]) : 0.f;
      h[c] = fmaf(p.beta, zx[c], x[c]);
    }
    if (valid) {
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        __stcs(st_h + (ih + c * Tp), make_float2(zx[2 * c], zx[2 * c + 1]));
        __stcs(st_h + (ih + (3 + c) * Tp), act ? make_float2(x[2 * c], x[2 * c + 1]) : make_float2(0.f, 0.f));
      }
    }
  } else {
#pragma unroll
    for (int c = 0; c < 6; ++c) h[c] = x[c];
  }
  float2* const b2 = reinterpret_cast<float2*>(bufB);  // [3][TS_BLOCK] channel pairs
#pragma unroll
  for (int c = 0; c < 3; ++c) b2[c * TS_BLOCK + tid] = make_float2(h[2 * c], h[2 * c + 1]);
  // S8d drift draws (Eq. 25): Philox streams 0 / 1 -> six normals (before the barrier: independent work)
  float z[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  if (act) {
    const uint32_t nstep = p.gstep - __ldg(p.reset_step + e);
    const uint4 w0 = philox4x32_10(make_uint4(env, (uint32_t)j, nstep, ep4 | 0u), p.seed_lo, p.seed_hi);
    const uint4 w1 = philox4x32_10(make_uint4(env, (uint32_t)j, nstep, ep4 | 1u), p.seed_lo, p.seed_hi);
    box_muller(w0.x, w0.y, z[0], z[1]);
    box_muller(w0.z, w0.w, z[2], z[3]);
    box_muller(w1.x, w1.y, z[4], z[5]);
  }
  float zw[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};  // Eq. 25 white noise n_t / sigma (R3): streams 6 / 7
  if (EXT && act && (p.sigma_wf != 0.f || p.sigma_wt != 0.f)) {
    const uint32_t nstep = p.gstep - __ldg(p.reset_step + e);
    const uint4 w0 = philox4x32_10(make_uint4(env, (uint32_t)j, nstep, ep4 | 6u), p.seed_lo, p.seed_hi);
    const uint4 w1 = philox4x32_10(make_uint4(env, (uint32_t)j, nstep, ep4 | 7u), p.seed_lo, p.seed_hi);
    box_muller(w0.x, w0.y, zw[0], zw[1]);
    box_muller(w0.z, w0.w, zw[2], zw[3]);
    box_muller(w1.x, w1.y, zw[4], zw[5]);
  }
  __syncthreads();
  if (TS_HYST_STORE_LATE && MODE == TS_HYST_ASYM && valid) {
#pragma unroll
    for (int c = 0; c < 3; ++c) __stcs(st_h + (ih + c * Tp), make_float2(h[2 * c], h[2 * c + 1]));
  }
  // S8c crosstalk (D4): c_j = h_j + chi/4 sum_{k in N4(j)} (h_k - h_j); a missing neighbour is
  // replaced by the taxel itself (h_j - h_j = 0), so the sum needs no predicates.
  const int nu = (meta >> 8) & 255;  // slots of a patch are consecutive: -u/+u = tid -/+ 1, -v/+v = tid -/+ nu
  const int n0 = (meta & (1 << 16)) ? tid - 1 : tid, n1 = (meta & (1 << 17)) ? tid + 1 : tid;
  const int n2 = (meta & (1 << 18)) ? tid - nu : tid, n3 = (meta & (1 << 19)) ? tid + nu : tid;
  const float q4 = 0.25f * p.chi;
  float outv[6], Dn[6], nsum[6];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const float2* hb = b2 + c * TS_BLOCK;
    const float2 a0 = hb[n0], a1 = hb[n1], a2 = hb[n2], a3 = hb[n3];
    nsum[2 * c] = (a0.x + a1.x) + (a2.x + a3.x);
    nsum[2 * c + 1] = (a0.y + a1.y) + (a2.y + a3.y);
  }
  // Eq. 11 / 31 with the Gaussian kernel (R7): conv = sum_{du,dv} g[|du|] g[|dv|] h(iu+du, iv+dv), zero outside the
  // patch; slots of a patch are consecutive (u fastest), inactive sources hold h = 0.  The kernel is separable, so the
  // sum runs as two 1-D passes through the exchange buffer, (2r+1) + (2r+1) taps instead of (2r+1)^2: row sums
  // t(iu, iv) = sum_du g[|du|] h(iu+du, iv) replace h in the buffer (two barriers; `gauss` is block-uniform), then
  // conv = sum_dv g[|dv|] t(iu, iv+dv).  A patch is active or filtered as a whole (the link filter works per link, R_j per
  // patch), so the row sums a column pass reads were all formed.
  float conv[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  const bool gauss = EXT && p.xt_r > 0;
  if (gauss) {
    const int r = p.xt_r;
    int nv = 0, iv = 0, iu = 0;
    float t6[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    if (act) {
      const TsPatch& pt = p.patches[patch0 + (meta & 255)];
      nv = __ldg(&pt.nv);
      const int il = j - __ldg(&pt.start);
      iv = il / nu; iu = il - iv * nu;
      for (int du = -r; du <= r; ++du) {
        if (iu + du < 0 || iu + du >= nu) continue;
        const float w = p.xt_w[du < 0 ? -du : du];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const float2 a = b2[c * TS_BLOCK + tid + du];
          t6[2 * c] = fmaf(w, a.x, t6[2 * c]);
          t6[2 * c + 1] = fmaf(w, a.y, t6[2 * c + 1]);
        }
      }
    }
    __syncthreads();   // every row pass has read h
#pragma unroll
    for (int c = 0; c < 3; ++c) b2[c * TS_BLOCK + tid] = make_float2(t6[2 * c], t6[2 * c + 1]);
    __syncthreads();
    if (act) {
      for (int dv = -r; dv <= r; ++dv) {
        if (iv + dv < 0 || iv + dv >= nv) continue;
        const float w = p.xt_w[dv < 0 ? -dv : dv];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const float2 a = b2[c * TS_BLOCK + tid + dv * nu];
          conv[2 * c] = fmaf(w, a.x, conv[2 * c]);
          conv[2 * c + 1] = fmaf(w, a.y, conv[2 * c + 1]);
        }
      }
    }
  }
  float cxv[6];
  if (gauss) {
#pragma unroll
    for (int c = 0; c < 6; ++c) cxv[c] = fmaf(p.chi, conv[c], (1.f - p.chi) * h[c]);
  } else {
#pragma unroll
    for (int c = 0; c < 3; ++c) {  // channel pairs: two FFMA2 per pair
      const float2 h2 = make_float2(h[2 * c], h[2 * c + 1]);
      const float2 acc = fma2(bc2(-4.f), h2, make_float2(nsum[2 * c], nsum[2 * c + 1]));  // sum_k (h_k - h_j)
      const float2 cx = fma2(bc2(q4), acc, h2);
      cxv[2 * c] = cx.x; cxv[2 * c + 1] = cx.y;
    }
  }
  // Eq. 25 read delay (R9): the readout of step n shows the post-crosstalk signal of step n - Delta_n,
  // Delta_n = max(0, Delta + k_n), k_n uniform on {-J..J}, one draw per (env, step): stream 9, taxel counter
  // 0xffffffff.  The ring holds the fields of the last S = Delta + J steps; step n lives in slot n mod S, which is
  // also the slot of step n - S, so the read comes first; the write is issued at the very end of the chain, after
  // the loaded values have been consumed: a store to a line whose read miss is still outstanding cost 0.9 ms per
  // step on config 5 (2.65 -> 1.9 ms, measured).  A slot is only read for a step >= 0 of the current episode
  // (earlier ones read 0, Q12), hence no clearing at reset.
  const bool ring_on = EXT && p.rd_S > 0 && valid;
  float2 ringw[3];
  unsigned iw = 0u;
  if (ring_on) {
    const uint32_t nstep = p.gstep - __ldg(p.reset_step + e);
    int delta = p.rd_delay;
    if (p.rd_jitter > 0) {
      const uint4 w = philox4x32_10(make_uint4(env, 0xffffffffu, nstep, ep4 | 9u), p.seed_lo, p.seed_hi);
      const int k = (int)(((unsigned long long)(w.x >> 9) * (unsigned long long)(2 * p.rd_jitter + 1)) >> 23) - p.rd_jitter;
      delta = max(0, p.rd_delay + k);
    }
    float2* const ring = reinterpret_cast<float2*>(p.st_ring);
    const unsigned S = (unsigned)p.rd_S;
    float2 dl[3] = {make_float2(cxv[0], cxv[1]), make_float2(cxv[2], cxv[3]), make_float2(cxv[4], cxv[5])};
    if (delta > 0) {
      const bool have = (uint32_t)delta <= nstep;
      const unsigned ir = (((unsigned)e * S + (nstep - (uint32_t)delta) % S) * 3u) * Tp + (unsigned)j;
#pragma unroll
      for (int c = 0; c < 3; ++c) dl[c] = have ? ld_stream2(ring + (ir + c * Tp)) : make_float2(0.f, 0.f);
    }
    iw = (((unsigned)e * S + nstep % S) * 3u) * Tp + (unsigned)j;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      ringw[c] = make_float2(cxv[2 * c], cxv[2 * c + 1]);
      cxv[2 * c] = dl[c].x; cxv[2 * c + 1] = dl[c].y;
    }
  }
#pragma unroll
  for (int c = 0; c < 6; ++c) {
    const float cx = cxv[c];
    Dn[c] = act ? fmaf(c < 3 ? p.sigma_f : p.sigma_t, z[c], ns.sD[c]) : 0.f;
    if (!EXT) {
      outv[c] = (act && !deadb) ? cx + Dn[c] : 0.f;  // S8a dead (Eq. 28, D5) last
    } else {
      float y = fmaf(c < 3 ? p.sigma_wf : p.sigma_wt, zw[c], cx + (c < 3 ? p.bias_f : p.bias_t)) + Dn[c];  // Eq. 25
      const float q = c < 3 ? p.quant_f : p.quant_t;
      if (q > 0.f) y = rintf(y / q) * q;  // quantize(., q): IEEE fp32 division, round half to even
      outv[c] = act ? y : 0.f;
    }
  }
  const bool stuck_on = p.stuck_lo_f != 0.f || p.stuck_hi_f != 0.f || p.stuck_lo_t != 0.f || p.stuck_hi_t != 0.f;
  if (EXT && deadb && !stuck_on) {
#pragma unroll
    for (int c = 0; c < 6; ++c) outv[c] = 0.f;  // D5: stuck at zero
  }
  if (EXT && deadb && stuck_on) {  // Eq. 28 stuck readout z_bj (R4): streams 4 / 5, n = 0; rare (p_dead of the taxels)
    const uint4 w0 = philox4x32_10(make_uint4(env, (uint32_t)j, 0u, ep4 | 4u), p.seed_lo, p.seed_hi);
    const uint4 w1 = philox4x32_10(make_uint4(env, (uint32_t)j, 0u, ep4 | 5u), p.seed_lo, p.seed_hi);
    const uint32_t ww[6] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y};
#pragma unroll
    for (int c = 0; c < 6; ++c) {
      const float lo = c < 3 ? p.stuck_lo_f : p.stuck_lo_t, hi = c < 3 ? p.stuck_hi_f : p.stuck_hi_t;
      outv[c] = fmaf(hi - lo, (float)(2u * (ww[c] >> 9) + 1u) * 5.9604644775390625e-8f, lo);
    }
  }
  if (valid) {
#pragma unroll
    for (int c = 0; c < 3; ++c) __stcs(st_d + (id + c * Tp), make_float2(Dn[2 * c], Dn[2 * c + 1]));
  }
  if ((FAST || p.ft_noisy) && valid) store6(p.ft_noisy + ej * 6u, outv);
  if (ring_on) {
#pragma unroll
    for (int c = 0; c < 3; ++c) __stcs(reinterpret_cast<float2*>(p.st_ring) + (iw + c * Tp), ringw[c]);
  }
}

// Stand-alone noise kernel (split variant): reads the clean ft the geometry kernel wrote.
template <int HM>
__global__ void __launch_bounds__(TS_BLOCK, 6) ts_noise_kernel(const __grid_constant__ TsStepParams p) {
  __shared__ float bufB[6 * TS_BLOCK];
  const int tid = threadIdx.x;
  const int e = blockIdx.x;
  const int4 g0 = __ldg(reinterpret_cast<const int4*>(p.groups + blockIdx.y));
  const int gstart = g0.x, gcount = g0.y;
  const bool valid = tid < gcount;
  const int j = gstart + (valid ? tid : 0);
  const unsigned ej = (unsigned)e * (unsigned)p.T + (unsigned)j;  // < 2^32 / 12 (checked by ts_create)
  NoiseState ns;
  noise_load<HM>(p, e, j, valid, ns);
  float ft[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  bool act = false, deadb = false;
  if (valid) {
    const float2* f2 = reinterpret_cast<const float2*>((p.ft_pert ? p.ft_pert : p.ft) + ej * 6u);  // ft_pert: Eq. 26 readout
    const float2 a = __ldcs(f2), b = __ldcs(f2 + 1), c = __ldcs(f2 + 2);
    ft[0] = a.x; ft[1] = a.y; ft[2] = b.x; ft[3] = b.y; ft[4] = c.x; ft[5] = c.y;
    act = __ldg(&p.tx_pos[j].w) > 0.f;
    deadb = act && ((p.st_flags[ej] >> 1) & 1);
  }
  noise_chain<HM>(p, e, j, ej, tid, g0.z, valid, act, deadb, valid ? __ldg(p.tx_meta + j) : 0, ft, ns, bufB);
  if (p.clock && tid == 0) atomicMax(p.clock + 1, globaltimer_ns());   // device-side clock: the split form ends the step here
}

template <bool SINGLE, bool FAST = false>
__device__ __forceinline__ void march_phase(const TsStepParams& p, const FrameS* frames, int e, int lp, bool valid, bool act,
                                            unsigned ej, float phif, F3 xo, float4 P4, int pidx) {
// ---- phase 2 (S7): proximity march, t <- min(t + max(phi(q + t a), 0), r_prox), K_m evaluations.
  // Exact shortcuts (O7): evaluation 0 is the query above; t = r_prox is absorbing; an evaluation
  // that leaves t unchanged repeats forever.
  if (FAST || p.prox) {
    float t = 0.f;
    int go = 0;  // int, not bool: a bool that lives across the loop is packed into a byte and costs PRMTs
    if (act && p.march_steps > 0) {
      t = fminf(fmaxf(phif, 0.f), p.r_prox);
      go = (t > 0.f) && (t < p.r_prox);
    }
    if (SINGLE) {
      const FrameS& F = frames[lp];
      const int gtype = __ldg(p.g_type + e);  // block-uniform (one object per env)
      const F3 dr = mk3(F.dirf[0], F.dirf[1], F.dirf[2]);  // M n of the patch normal, built with the frame
      if (gtype == TS_GEOM_SDF) {
        const int N = p.grid_n;
        const float4* bank_g = p.bank + (size_t)(int)F.prm[0] * p.grid_stride;
        const float half = 0.5f * (float)(N - 1);
        const F3 u0 = mk3(fmaf(xo.x, p.inv_voxel, half), fmaf(xo.y, p.inv_voxel, half), fmaf(xo.z, p.inv_voxel, half));
        const F3 du = p.inv_voxel * dr;
        const F3 u1 = u0 + p.r_prox * du;
        const float lo = 0.75f, hi = (float)N - 1.75f;
        const bool inside = fminf(fminf(fminf(u0.x, u0.y), u0.z), fminf(fminf(u1.x, u1.y), u1.z)) >= lo &&
                            fmaxf(fmaxf(fmaxf(u0.x, u0.y), u0.z), fmaxf(fmaxf(u1.x, u1.y), u1.z)) <= hi;
        if (__all_sync(TS_FULL, inside || !go)) {  // whole segment inside the grid for every marching lane
          const unsigned cbase = (unsigned)(int)F.prm[0] * (unsigned)p.grid_stride -
                                 0x4B400000u * (unsigned)((N - 1) * N + N + 1);
          // Interior points (u in [0.75, N-1.75]): floor by a round-down add of 1.5*2^23 (ulp 1 there, so the
          // sum is floor(u) + 1.5*2^23 exactly; FADDs on the FMA pipe instead of F2I/I2F on the quarter-rate
          // conversion pipe).  The three 0x4B400000 biases of the integer images and the grid offset are
          // folded into `cbase` (32-bit wrap-around arithmetic): two IMADs and one add per cell index.
          // A converging ray takes sub-voxel steps, so consecutive evaluations mostly fall into the same cell:
          // its 8 corners stay in registers and are reloaded only when the cell index changes.
          unsigned pidx = 0xffffffffu;
          float4 A = make_float4(0.f, 0.f, 0.f, 0.f), B = A;
          // No per-lane "finished" state inside the loop: every exit of O7 is a fixed point of the update (t = cap
          // stays at cap; an evaluation that left t unchanged is repeated at the same point and leaves it unchanged
          // again), so a finished lane simply keeps evaluating and t does not move.  Lanes that never march get their own
          // cap = t (and never gather: their segment may leave the bank; A = B = 0 gives s = 0).  Only the loop exit
          // looks at the lanes: one vote on "t moved and is below the cap".  Against the form with a per-lane flag this
          // drops the FSEL / SEL / 3 ISETP of every iteration (5 of 45 instructions); same t, bit for bit.
          const bool m0 = go != 0;
          const float cap = m0 ? p.r_prox : t;
          bool cont = __any_sync(TS_FULL, m0);
          for (int left = p.march_steps - 1; left > 0 && cont; --left) {   // down-counter: no re-read of march_steps
            const F3 u = u0 + t * du;
            const float MAGIC = 12582912.f;  // 1.5 * 2^23
            const float tx = __fadd_rd(u.x, MAGIC), ty = __fadd_rd(u.y, MAGIC), tz = __fadd_rd(u.z, MAGIC);
            const unsigned idx = ((__float_as_uint(ty) * (unsigned)(N - 1) + __float_as_uint(tx)) * (unsigned)N + __float_as_uint(tz)) + cbase;
            if (m0 && idx != pidx) {
              A = __ldg(p.bank + idx);
              B = __ldg(p.bank + idx + 1);
              pidx = idx;
            }
            const float sv = trilerp(A, B, u.x - (tx - MAGIC), u.y - (ty - MAGIC), u.z - (tz - MAGIC));
            const float tn = fminf(t + fmaxf(sv, 0.f), cap);
            cont = __any_sync(TS_FULL, (tn != t) && (tn < cap));
            t = tn;
          }
        } else {
          for (int it = 1; it < p.march_steps; ++it) {
            if (!__any_sync(TS_FULL, go)) break;
            if (go) {
              const float sv = grid_value_f(p, bank_g, u0 + t * du);
              const float tn = fminf(t + fmaxf(sv, 0.f), p.r_prox);
              go = (tn != t) && (tn < p.r_prox);
              t = tn;
            }
          }
        }
      } else {
        // same fixed-point form as the grid loop: lanes that never march carry cap = t
        const float cap = go ? p.r_prox : t;
        bool cont = __any_sync(TS_FULL, go);
#define TS_PRIM_LOOP(TYPE)                                                         \
  for (int left = p.march_steps - 1; left > 0 && cont; --left) {                   \
    const float sv = prim_value_f(TYPE, F.prm, xo + t * dr);                       \
    const float tn = fminf(t + fmaxf(sv, 0.f), cap);                               \
    cont = __any_sync(TS_FULL, (tn != t) && (tn < cap));                           \
    t = tn;                                                                        \
  }
        if (gtype == TS_GEOM_SPHERE) { TS_PRIM_LOOP(TS_GEOM_SPHERE) }
        else if (gtype == TS_GEOM_BOX) { TS_PRIM_LOOP(TS_GEOM_BOX) }
        else if (gtype == TS_GEOM_CAPSULE) { TS_PRIM_LOOP(TS_GEOM_CAPSULE) }
#undef TS_PRIM_LOOP
      }
    } else {
      const F3 xj = mk3(P4.x, P4.y, P4.z);
      const float4 na = __ldg(&p.patches[pidx].na);
      const F3 nj = mk3(na.x, na.y, na.z);
      for (int it = 1; it < p.march_steps; ++it) {
        if (!__any_sync(TS_FULL, go)) break;
        if (go) {
          const F3 y = xj + t * nj;
          float sv = __int_as_float(0x7f800000);
          for (int k = 0; k < p.K; ++k) {
            const FrameS& F = frames[lp * p.K + k];
            // fp32 images of M and c, rounded here (K > 1 only; the single-object path marches from xo and dirf)
            const float m0 = (float)F.M[0], m1 = (float)F.M[1], m2 = (float)F.M[2], m3 = (float)F.M[3], m4 = (float)F.M[4],
                        m5 = (float)F.M[5], m6 = (float)F.M[6], m7 = (float)F.M[7], m8 = (float)F.M[8];
            const F3 x = mk3((float)F.c[0] + fmaf(m0, y.x, fmaf(m1, y.y, m2 * y.z)), (float)F.c[1] + fmaf(m3, y.x, fmaf(m4, y.y, m5 * y.z)),
                             (float)F.c[2] + fmaf(m6, y.x, fmaf(m7, y.y, m8 * y.z)));
            sv = fminf(sv, phi_f(p, F.type, F.prm, x));
          }
          const float tn = fminf(t + fmaxf(sv, 0.f), p.r_prox);
          go = (tn != t) && (tn < p.r_prox);
          t = tn;
        }
      }
    }
    if (valid) __stcs(p.prox + ej, act ? p.r_prox - t : 0.f);
  }
}

// HM = TS_HYST_* of the fused noise chain, -1 = no noise chain in this kernel.  FAST = the common full configuration
// fixed at compile time: every output pointer given, group records in the parameter space, env order table present,
// DMMA marker path.  The generic variant tests each of these per block (a 64-bit pointer test per output, both group
// record paths issued under predicates): ~35 issue slots per warp that FAST does not spend.
template <bool SINGLE, int HM, bool FAST = false>
__global__ void __launch_bounds__(TS_BLOCK, TS_MIN_BLOCKS) ts_step_kernel(const __grid_constant__ TsStepParams p) {
  constexpr bool NOISE = HM >= 0;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  // Shared memory is kept small on purpose: it is carved out of the same 256 KB as L1, and the SDF gathers
  // of the march live on L1 hits.  S (marker phase) aliases bufB (noise phase); a barrier separates them.
  // Fixed-size arrays first, at compile-time offsets (their addresses are re-formed at every use under the 48-register
  // budget: an immediate instead of arithmetic on kernel parameters); the frames, whose count is the layout's, last.
  float* hh = reinterpret_cast<float*>(smem_raw);         // [TS_BLOCK] penetration h_i (Eq. 19)
  float* ha = hh + TS_BLOCK;                              // [TS_BLOCK] h_i^alpha_e
  unsigned* pmask = reinterpret_cast<unsigned*>(ha + TS_BLOCK);  // bit l: group-local patch l has penetration
  double* S = reinterpret_cast<double*>(smem_raw + sizeof(float) * 2 * TS_BLOCK + sizeof(int) * TS_MAX_GROUP_PATCHES);
                                                          // [3][TS_CHUNK] marker pass-1 sums (generic marker path only)
  float* bufB = reinterpret_cast<float*>(S);              // [6][TS_BLOCK] crosstalk exchange (first 6 KB of S)
  FrameS* frames = reinterpret_cast<FrameS*>(reinterpret_cast<unsigned char*>(S) +
                                             (FAST ? (int)(sizeof(float) * 6 * TS_BLOCK) : p.s_bytes));   // FAST implies the DMMA marker path

  const int tid = threadIdx.x;
#if TS_GRID_GFAST
  // grid (G, min(E, 65535), ceil(E / 65535)): the group index runs fastest, and no integer division is needed
  const unsigned bxi = blockIdx.z * 65535u + blockIdx.y;
  const int gi = (int)blockIdx.x;
  if (bxi >= (unsigned)p.E) return;
#else
  const unsigned bxi = blockIdx.x;
  const int gi = blockIdx.y;
#endif
  const int e = (FAST || p.env_perm) ? __ldg(p.env_perm + bxi) : (int)bxi;
  int gstart, gcount, patch0, npatch, chunk0, nchunk, gmcount;
  if (FAST || p.inl) {  // group record from the parameter space (constant bank)
    const TsGroup& g = p.inl_grp[gi];
    gstart = g.start; gcount = g.count; patch0 = g.patch0; npatch = g.npatch; chunk0 = g.chunk0; nchunk = g.nchunk; gmcount = g.mcount;
  } else {
    const int4 g0 = __ldg(reinterpret_cast<const int4*>(p.groups + gi));
    const int4 g1 = __ldg(reinterpret_cast<const int4*>(p.groups + gi) + 1);
    gstart = g0.x; gcount = g0.y; patch0 = g0.z; npatch = g0.w; chunk0 = g1.x; nchunk = g1.y; gmcount = g1.w;
  }

  // ---- phase 0: this block's relative poses arrive from frames_g (ts_frames_kernel) by ONE bulk copy (TMA) ------
  __shared__ __align__(8) uint64_t fbar;
  if (tid == 0) {
    *pmask = 0u;
    mbar_init(&fbar, 1);
    const unsigned bytes = (unsigned)(npatch * p.K) * (unsigned)sizeof(FrameS);
    mbar_expect_tx(&fbar, bytes);
    const FrameS* src = reinterpret_cast<const FrameS*>(p.frames_g) + ((size_t)bxi * p.P + patch0) * p.K;
#if TS_PDL
    // Programmatic dependent launch: this grid may start while ts_frames_kernel is still draining.  This thread reads
    // frames_g (through the bulk copy below), so it waits for the frames grid to complete and flush.  (With TS_PDL = 1
    // it is the only thread that has to: the previous step kernel finished before the frames kernel began.  With the
    // chained launch of TS_PDL = 2 every thread waits again below, before it reads state.)
    asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
    bulk_g2s(frames, src, bytes, &fbar);
    // L2 prefetch of the same rows for the block TS_PF_AHEAD positions later in launch order (blockIdx.x runs fastest):
    // by the time that block starts, its bulk copy is an L2 hit instead of a DRAM round trip in front of phase 1.
    constexpr unsigned AH = TS_GRID_GFAST ? TS_PF_AHEAD / 4 : TS_PF_AHEAD;
    if (TS_PF_AHEAD > 0 && bxi + AH < (unsigned)p.E)
      asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src + (size_t)AH * p.P * p.K), "r"(bytes) : "memory");
#if TS_STATE_BULK_PF == 1
    if (NOISE) noise_prefetch_bulk<HM>(p, e, gstart, gcount);
#endif
  }
  const bool valid = tid < gcount;
  const int j = gstart + (valid ? tid : 0);
  const unsigned ej = (unsigned)e * (unsigned)p.T + (unsigned)j;  // < 2^32 / 12 (checked by ts_create)
  const float4 P4 = __ldg(p.tx_pos + j);
  const int meta = valid ? __ldg(p.tx_meta + j) : 0;  // idle threads: no neighbours, patch 0
  const int lp = meta & 255;
  const float Rj = valid ? P4.w : 0.f;  // R_j = 0: inactive slot
  const bool act = Rj > 0.f;
#if TS_PDL >= 2
  // Every thread: the flag byte and the state rows read below were written by the PREVIOUS step kernel.  With the
  // chained launch this grid's blocks can be resident before that kernel has finished; it is complete once the frames
  // grid in front of this one is (whose blocks waited for it at their top).
  asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
  uint8_t flag = valid ? p.st_flags[ej] : (uint8_t)0;
#if TS_STATE_BULK_PF == 0
  if (NOISE) noise_prefetch<HM>(p, e, gstart + (tid & ~31), gstart + gcount, tid & 31);
#endif
  __syncthreads();        // publishes the mbarrier (and pmask); every warp arrives within a few cycles of block start
  mbar_wait(&fbar, 0u);   // frames landed in shared memory (async-proxy writes are visible after the wait)
#if TS_PDL >= 2
  // This block no longer needs frames_g: once every block of the grid has said so, the next step's frames kernel may
  // start overwriting it (it then runs alongside this grid's last wave).
  asm volatile("griddepcontrol.launch_dependents;");
#endif

  // ---- phase 1 (S1-S4): x_o = c + M x_j, phi = min_k phi_k, depth (Eq. 2), contact (Eq. 3) ----
  double phid = __longlong_as_double(0x7ff0000000000000LL);
  D3 xd = D3{0.0, 0.0, 0.0};
  int kst = 0;
  if (act) {
    const D3 xj = D3{(double)P4.x, (double)P4.y, (double)P4.z};
    for (int k = 0; k < (SINGLE ? 1 : p.K); ++k) {
      const FrameS& F = frames[lp * (SINGLE ? 1 : p.K) + k];
      const D3 x = ldv(F.c) + mulR(F.M, xj);
      const double ph = phi_d(p, F.type, F.prm, x);
      if (SINGLE) {  // one object: no comparison (and none of its 8 predicated register moves)
        phid = ph; xd = x;
      } else if (ph < phid) {  // strict: ties -> lowest k (Q3)
        phid = ph; kst = k; xd = x;
      }
    }
  }
  const float phif = (float)phid;
  float d = 0.f;
  if (act) {
    const double dd = (double)Rj - phid;
    d = dd > 0.0 ? (float)dd : 0.f;
  }
  const bool yb = act && ((d > p.eta_on) || ((flag & 1) && d > p.eta_off));
  const bool deadb = p.noise_enable && act && ((flag >> 1) & 1);
  if (valid) {
    p.st_flags[ej] = (uint8_t)((flag & 2) | (yb ? 1 : 0));  // Schmitt state from the un-masked bit (O4)
    if (FAST || p.contact) p.contact[ej] = (yb && !deadb) ? 1 : 0;
    if ((FAST && NOISE) || p.dead) p.dead[ej] = deadb ? 1 : 0;
    if (FAST || p.depth) __stcs(p.depth + ej, d);
  }
  if (FAST || p.marker) {  // Eq. 19: h_i = max(0, -phi), no R_j
    const float h = (act && phid < 0.0) ? (float)(-phid) : 0.f;
    hh[tid] = h;
    ha[tid] = h > 0.f ? __powf(h, p.alpha_e) : 0.f;
    const unsigned wb = __reduce_or_sync(TS_FULL, h > 0.f ? (1u << lp) : 0u);  // one shared atomic per warp
    if ((tid & 31) == 0 && wb) atomicOr(pmask, wb);
  }
  const F3 xo = mk3((float)xd.x, (float)xd.y, (float)xd.z);  // fp32 object-frame position for the march

#if !TS_MARCH_LATE
  march_phase<SINGLE, FAST>(p, frames, e, lp, valid, act, ej, phif, xo, P4, patch0 + lp);
#endif

  // ---- phase 3 (S5): kinematic force / torque (Eq. 4-9, D2) in double, link frame ---------------
  // Eq. 26 (R8): the noisy readout senses with R~_j = max(0, R_j + eps_j), eps_j ~ U[-rho, rho] drawn once per
  // (env, taxel, episode) from stream 8, n = 0, word 0; dn = [R~_j - phi]_+ is the depth the noise chain starts
  // from.  Only the variants that carry the remaining A.8 knobs (and the two-kernel variant) evaluate it.
  constexpr bool RN = HM < 0 || (HM & 4) != 0;
  const bool rn_on = RN && p.rho != 0.f;  // block-uniform
  float dn = d;
  if (rn_on && act) {
    const uint4 w = philox4x32_10(make_uint4(p.env_id_base + (uint32_t)e, (uint32_t)j, 0u, (__ldg(p.episode + e) << 4) | 8u), p.seed_lo, p.seed_hi);
    const double u = (double)(2u * (w.x >> 9) + 1u) * 5.9604644775390625e-8;
    const double Rt = fmax(0.0, (double)Rj + fma(2.0 * (double)p.rho, u, -(double)p.rho));
    const double dd = Rt - phid;
    dn = dd > 0.0 ? (float)dd : 0.f;
  }
  if (RN && p.depth_pert && valid) __stcs(p.depth_pert + ej, dn);   // input of the noisy depth readout (R10)
  float ft[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  float fn6[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};  // Eq. 4-9 at depth dn (dead code unless rn_on)
  const bool touch = d > 0.f || (rn_on && dn > 0.f);
  if ((FAST || p.ft != nullptr || NOISE || rn_on) && __any_sync(TS_FULL, touch)) {
    if (touch) {  // Q5: every term gated on d > 0
      const FrameS& F = frames[lp * (SINGLE ? 1 : p.K) + kst];
      const D3 g = grad_d(p, F.type, F.prm, xd);
      const double g2 = dot(g, g);
      D3 mbar;  // contact normal in the link frame, m_bar = R_L^T m = M^T g / |g|
      if (g2 < 1e-24) {  // Q2: m = -a_j, i.e. minus the patch normal in the link frame
        const float4 na = __ldg(&p.patches[patch0 + lp].na);
        mbar = D3{-(double)na.x, -(double)na.y, -(double)na.z};
      }
      else mbar = drsqrt_n(g2) * mulRT(F.M, g);
      const D3 x = D3{(double)P4.x, (double)P4.y, (double)P4.z};
      // Everything but the depth is shared by the clean readout (depth d) and the Eq. 26 one (depth dn).
      if (!RN) {
        // Variants without Eq. 26 (compile-time): one readout, written straight through.  The shared form below
        // costs this variant 0.6 % of the step on config 5 (different register allocation), measured.
        const double sj = (double)__powf(d, p.alpha);  // s_j = d^alpha
        D3 f, tau;
        if (p.use_velocity) {
          const D3 wO = ldv(F.wO), wL = ldv(F.wL);
          const D3 vrel = ldv(F.vbar) + cross(wO, ldv(F.cbar) + x) - cross(wL, x);     // Eq. 4-6
          const double vns = dot(vrel, mbar);
          const D3 vt = vrel - vns * mbar;                                             // Eq. 7
          const double fnm = sj * fma((double)p.c_n, vns, (double)p.k_n);
          D3 ftan = (-(double)p.k_t) * vt;                                             // Eq. 8 tangential
          const double lim = (double)p.mu * fabs(fnm), nft2 = dot(ftan, ftan);
          if (nft2 > lim * lim) ftan = (lim * drsqrt_n(nft2)) * ftan;                  // D2 Coulomb cap
          f = fnm * mbar + ftan;
          tau = cross(x, f) - ((double)p.k_omega * dot(wO - wL, mbar)) * mbar;         // Eq. 9
        } else {
          f = ((double)p.k_n * sj) * mbar;
          tau = cross(x, f);
        }
        ft[0] = (float)f.x; ft[1] = (float)f.y; ft[2] = (float)f.z;
        ft[3] = (float)tau.x; ft[4] = (float)tau.y; ft[5] = (float)tau.z;
      } else if (p.use_velocity) {
        const D3 wO = ldv(F.wO), wL = ldv(F.wL);
        const D3 vrel = ldv(F.vbar) + cross(wO, ldv(F.cbar) + x) - cross(wL, x);       // Eq. 4-6
        const double vns = dot(vrel, mbar);
        const D3 vt = vrel - vns * mbar;                                               // Eq. 7
        const D3 ftan0 = (-(double)p.k_t) * vt;                                        // Eq. 8 tangential
        const double nft2 = dot(ftan0, ftan0);
        const double spin = (double)p.k_omega * dot(wO - wL, mbar);
        auto readout = [&](float dep, float* o) {
          const double fnm = (double)__powf(dep, p.alpha) * fma((double)p.c_n, vns, (double)p.k_n);  // s_j = d^alpha
          D3 ftan = ftan0;
          const double lim = (double)p.mu * fabs(fnm);
          if (nft2 > lim * lim) ftan = (lim * drsqrt_n(nft2)) * ftan;                  // D2 Coulomb cap
          const D3 f = fnm * mbar + ftan;
          const D3 tau = cross(x, f) - spin * mbar;                                    // Eq. 9
          o[0] = (float)f.x; o[1] = (float)f.y; o[2] = (float)f.z;
          o[3] = (float)tau.x; o[4] = (float)tau.y; o[5] = (float)tau.z;
        };
        if (d > 0.f) readout(d, ft);
        if (rn_on && dn > 0.f) readout(dn, fn6);
      } else {
        auto readout = [&](float dep, float* o) {
          const D3 f = ((double)p.k_n * (double)__powf(dep, p.alpha)) * mbar;
          const D3 tau = cross(x, f);
          o[0] = (float)f.x; o[1] = (float)f.y; o[2] = (float)f.z;
          o[3] = (float)tau.x; o[4] = (float)tau.y; o[5] = (float)tau.z;
        };
        if (d > 0.f) readout(d, ft);
        if (rn_on && dn > 0.f) readout(dn, fn6);
      }
    }
  }
  if ((FAST || p.ft) && valid) store6(p.ft + ej * 6u, ft);
  if (rn_on) {  // from here on only the Eq. 26 readout is needed
#pragma unroll
    for (int c = 0; c < 6; ++c) ft[c] = fn6[c];
    if (HM < 0 && p.ft_pert && valid) store6(p.ft_pert + ej * 6u, ft);  // two-kernel variant: input of ts_noise_kernel
  }

  // ---- phase 4 (S8): noise chain (fused variant); contains the barrier that also publishes hh / ha / pact
  NoiseState ns;
  if (NOISE) noise_load<HM>(p, e, j, valid, ns);
  if (NOISE) noise_chain<HM, FAST>(p, e, j, ej, tid, patch0, valid, act, deadb, meta, ft, ns, bufB);
  else __syncthreads();
#if TS_MARCH_LATE
  march_phase<SINGLE, FAST>(p, frames, e, lp, valid, act, ej, phif, xo, P4, patch0 + lp);
#endif

  // ---- phase 5 (S6): elastomer marker dilation (Eq. 18-21, 23 first sum) ----------------------
  // With c = 1 and planar regular grids, g(r_ij) = exp(-lambda |r|^2) = gu(a,p) gv(b,q) and
  // r_ij = du(a,p) u^ + dv(b,q) v^, so u_j = s_d [ (u^ Uu + v^ Uv)/g_bar + n Un ] with
  //   pass 1 over (a,q): S0 = sum_p gu h, S1 = sum_p du gu h, T0 = sum_p gu h^alpha_e
  //   pass 2 over (a,b): Uu = sum_q gv S1, Uv = sum_q dv gv S0, Un = sum_q gv T0.
  // Sources with h_i = 0 contribute exactly 0; patches without penetration are skipped.
  if ((FAST || (p.marker && p.mk_mma)) && gmcount > 0) {
    // DMMA path (every patch fits 8 x 8 tiles): ONE WARP PER PATCH evaluates both passes as FP64 tensor-core products
    // (mma.m8n8k4, SASS DMMA.8x8x4) on zero-padded 8 x 8 tables; lane = 4 g + m holds A[row g][k m], B[k m][col g]
    // and C[row g][cols 2m, 2m+1].
    //   pass 1 (k = p):  S0 = GU H^T, S1 = DU H^T, T0 = GU Ha^T        with H[q][p] = h_i, C = S[a = g][q = 2m, 2m+1]
    //   pass 2 (k = q):  Uu = S1 GV^T, Uv = S0 DV^T, Un = T0 GV^T       contraction order q = 2m + kk, so that the A
    //                    operand of k-step kk is exactly the C element kk this lane already holds (no exchange).
    // hh / ha / pmask were published by the barrier above; no shared-memory scratch and no further barrier.
    const int lane = tid & 31, g = lane >> 2, m = lane & 3;
    const unsigned pm = *pmask;
    for (int l = tid >> 5; l < npatch; l += TS_BLOCK / 32) {
      const TsPatch& pt = p.patches[patch0 + l];
      const int mnu = __ldg(&pt.mnu), mnv = __ldg(&pt.mnv);
      if (mnu == 0) continue;
      float* o = p.marker + ((size_t)e * p.M + __ldg(&pt.mstart)) * 3;
      if (!((pm >> l) & 1u)) {  // no penetration anywhere in the patch: its markers are exactly 0
        for (int i = lane; i < mnu * mnv * 3; i += 32) __stcs(o + i, 0.f);
        continue;
      }
      const int nu = __ldg(&pt.nu), nv = __ldg(&pt.nv), base = __ldg(&pt.start) - gstart;
      const double* tab = p.mk_tab8 + (size_t)(patch0 + l) * 256;
      double s0a = 0.0, s0b = 0.0, s1a = 0.0, s1b = 0.0, t0a = 0.0, t0b = 0.0;
#pragma unroll
      for (int kk = 0; kk < 2; ++kk) {
        const int ip = kk * 4 + m;                    // B[k = p][n = q = g] = h[q][p]
        const bool ok = g < nv && ip < nu;
        const double h = ok ? (double)hh[base + g * nu + ip] : 0.0, hal = ok ? (double)ha[base + g * nu + ip] : 0.0;
        const double gu = __ldg(tab + g * 8 + ip), du = __ldg(tab + 64 + g * 8 + ip);   // A[a = g][k = p]
        dmma884(s0a, s0b, gu, h);
        dmma884(s1a, s1b, du, h);
        dmma884(t0a, t0b, gu, hal);
      }
      double uua = 0.0, uub = 0.0, uva = 0.0, uvb = 0.0, una = 0.0, unb = 0.0;
#pragma unroll
      for (int kk = 0; kk < 2; ++kk) {
        const double gv = __ldg(tab + 128 + g * 8 + 2 * m + kk), dv = __ldg(tab + 192 + g * 8 + 2 * m + kk);  // B[k = q][n = b = g]
        dmma884(uua, uub, kk ? s1b : s1a, gv);
        dmma884(uva, uvb, kk ? s0b : s0a, dv);
        dmma884(una, unb, kk ? t0b : t0a, gv);
      }
      const double sd = (double)p.s_d, kt = sd * p.inv_gbar;
      const float4 ua = __ldg(&pt.ua), va = __ldg(&pt.va), na = __ldg(&pt.na);
#pragma unroll
      for (int h2 = 0; h2 < 2; ++h2) {               // markers (a = g, b = 2m) and (a = g, b = 2m + 1)
        const int b = 2 * m + h2;
        if (g < mnu && b < mnv) {
          const double Uu = kt * (h2 ? uub : uua), Uv = kt * (h2 ? uvb : uva), Un = sd * (h2 ? unb : una);
          float* om = o + (b * mnu + g) * 3;
          __stcs(om, (float)fma(Uu, (double)ua.x, fma(Uv, (double)va.x, Un * (double)na.x)));
          __stcs(om + 1, (float)fma(Uu, (double)ua.y, fma(Uv, (double)va.y, Un * (double)na.y)));
          __stcs(om + 2, (float)fma(Uu, (double)ua.z, fma(Uv, (double)va.z, Un * (double)na.z)));
        }
      }
    }
  } else if (!FAST && p.marker && gmcount > 0) {
    // hh / ha / pact were completed by the barrier above; this one retires the crosstalk reads of bufB (= S)
    if (NOISE) __syncthreads();
    for (int ch = 0; ch < nchunk; ++ch) {
      const int4 c0 = __ldg(reinterpret_cast<const int4*>(p.chunks + chunk0 + ch));
      const int4 c1 = __ldg(reinterpret_cast<const int4*>(p.chunks + chunk0 + ch) + 1);
      const int i1b = c0.x, i1e = c0.y, mb = c0.z, me = c0.w, lpb = c1.x, lpe = c1.y;
      const unsigned pm = *pmask;
      const bool any = (pm & ((lpe >= 32 ? 0u : (1u << lpe)) - (1u << lpb))) != 0u;  // bits lpb .. lpe-1
      if (!any) {  // no penetration anywhere in the chunk: the markers are exactly 0
        float* o = p.marker + ((size_t)e * p.M + mb) * 3;
        for (int i = tid; i < (me - mb) * 3; i += TS_BLOCK) __stcs(o + i, 0.f);
        continue;
      }
      for (int it = tid; it < i1e - i1b; it += TS_BLOCK) {  // pass 1
        const int pk = __ldg(p.mk_item1 + i1b + it);
        const int l = pk & 255, a = (pk >> 8) & 255, q = pk >> 16;
        const TsPatch& pt = p.patches[patch0 + l];
        double s0 = 0.0, s1 = 0.0, t0 = 0.0;
        if ((pm >> l) & 1u) {
          const int nu = __ldg(&pt.nu);
          const double* GU = p.mk_tab + __ldg(&pt.tab) + a * nu;
          const double* DU = GU + __ldg(&pt.mnu) * nu;
          const int base = __ldg(&pt.start) - gstart + q * nu;
          for (int ip = 0; ip < nu; ++ip) {
            const double h = (double)hh[base + ip], hal = (double)ha[base + ip], gu = __ldg(GU + ip);
            s0 = fma(gu, h, s0);
            s1 = fma(__ldg(DU + ip), h, s1);
            t0 = fma(gu, hal, t0);
          }
        }
        S[it] = s0; S[TS_CHUNK + it] = s1; S[2 * TS_CHUNK + it] = t0;
      }
      __syncthreads();
      for (int im = tid; im < me - mb; im += TS_BLOCK) {  // pass 2: one marker per item
        float ox = 0.f, oy = 0.f, oz = 0.f;
        const int pk = __ldg(p.mk_item2 + mb + im);
        const int l = pk & 255, a = (pk >> 8) & 255, b = pk >> 16;
        const TsPatch& pt = p.patches[patch0 + l];
        if ((pm >> l) & 1u) {
          if (!__ldg(&pt.direct)) {
            const int nv = __ldg(&pt.nv), mnu = __ldg(&pt.mnu);
            const double* GV = p.mk_tab + __ldg(&pt.tab) + 2 * mnu * __ldg(&pt.nu) + b * nv;
            const double* DV = GV + __ldg(&pt.mnv) * nv;
            const double* s = S + (__ldg(&pt.i1off) - i1b + a);
            double Uu = 0.0, Uv = 0.0, Un = 0.0;
            for (int q = 0; q < nv; ++q) {
              const double gv = __ldg(GV + q);
              Uu = fma(gv, s[TS_CHUNK + q * mnu], Uu);
              Uv = fma(__ldg(DV + q), s[q * mnu], Uv);
              Un = fma(gv, s[2 * TS_CHUNK + q * mnu], Un);
            }
            const double sd = (double)p.s_d, kt = sd * p.inv_gbar;
            const float4 ua = __ldg(&pt.ua), va = __ldg(&pt.va), na = __ldg(&pt.na);
            ox = (float)(kt * fma(Uu, (double)ua.x, Uv * (double)va.x) + sd * Un * (double)na.x);
            oy = (float)(kt * fma(Uu, (double)ua.y, Uv * (double)va.y) + sd * Un * (double)na.y);
            oz = (float)(kt * fma(Uu, (double)ua.z, Uv * (double)va.z) + sd * Un * (double)na.z);
          } else {  // direct sum (c_e != 1: rho(r) = 1/(|r|^2 + eps^2) is not separable)
            const float4 mp = __ldg(p.mk_pos + mb + im), mn = __ldg(p.mk_nrm + mb + im);
            const D3 n = D3{(double)mn.x, (double)mn.y, (double)mn.z};
            const double eps = (double)pt.eps, ce = (double)p.c_e;
            D3 acc = D3{0.0, 0.0, 0.0};
            for (int i = 0; i < pt.n; ++i) {
              const float hi = hh[pt.start - gstart + i];
              if (!(hi > 0.f)) continue;
              const float4 xs = __ldg(p.tx_pos + pt.start + i);
              const D3 zv = D3{(double)mp.x - (double)xs.x, (double)mp.y - (double)xs.y, (double)mp.z - (double)xs.z};
              const D3 rr = zv - dot(zv, n) * n;                                     // Eq. 18
              const double r2 = dot(rr, rr);
              const double gg = exp(-(double)p.lambda_d * r2);
              const double w = (double)hi * (ce * gg * p.inv_gbar + (1.0 - ce) * (2.0 * eps) / (r2 + eps * eps));  // Eq. 20
              acc = acc + (double)p.s_d * (w * rr + ((double)ha[pt.start - gstart + i] * gg) * n);              // Eq. 21
            }
            ox = (float)acc.x; oy = (float)acc.y; oz = (float)acc.z;
          }
        }
        float* o = p.marker + ((size_t)e * p.M + mb + im) * 3;
        __stcs(o, ox); __stcs(o + 1, oy); __stcs(o + 2, oz);
      }
      if (ch + 1 < nchunk) __syncthreads();  // S is reused by the next chunk
    }
  }
  // device-side clock: last block end (thread 0 of every block; the fused form ends the step here)
  if (p.clock && tid == 0 && (NOISE || !p.noise_enable)) atomicMax(p.clock + 1, globaltimer_ns());
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
// stream 2 at n = 0, dead iff word0 < floor(p_dead 2^32).  One thread per (env, padded slot).
__global__ void ts_reset_state_kernel(const __grid_constant__ TsStepParams p, const uint8_t* mask, uint32_t thr, int nh) {
  const long long gt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gt >= (long long)p.E * p.Tp) return;
  const int e = (int)(gt / p.Tp), t = (int)(gt - (long long)e * p.Tp);
  if (mask && !mask[e]) return;
  if (p.st_hyst)
    for (int c = 0; c < nh; ++c) p.st_hyst[((size_t)e * nh + c) * p.Tp + t] = 0.f;
  if (p.st_drift)
    for (int c = 0; c < 6; ++c) p.st_drift[((size_t)e * 6 + c) * p.Tp + t] = 0.f;
  if (t >= p.T) return;
  uint8_t fl = 0;
  if (p.noise_enable && p.tx_pos[t].w > 0.f) {
    const uint4 w = philox4x32_10(make_uint4(p.env_id_base + (uint32_t)e, (uint32_t)t, 0u, (p.episode[e] << 4) | 2u), p.seed_lo, p.seed_hi);
    fl = (w.x < thr) ? 2 : 0;
  }
  p.st_flags[(size_t)e * p.T + t] = fl;
}

// ---------------------------------------------------------------------------------------
// R10: noisy readouts of the scalar sensors (Table 3: every knob of App. A.8 but crosstalk).
// One channel: x = gamma clean -> hysteresis -> y = h + b + sigma_w z_w + D (Eq. 25) -> quantize -> dead: stuck value.
// ---------------------------------------------------------------------------------------
template <int MODE>
__device__ __forceinline__ float scalar_chain(const TsStepParams& p, int cls, float clean, float gain, bool dead, float stuck_u,
                                              float z_rw, float z_w, float& ha, float& hb, float& drift, bool use_delayed,
                                              float delayed, float& hrec) {
  const float x = gain * clean;
  float h = x;
  if (MODE == TS_HYST_MAXWELL) {            // Eq. 29-30
    const float xi = fmaf(p.decay, ha, x - hb);
    ha = xi; hb = x;
    h = fmaf(p.beta, xi, x);
  } else if (MODE == TS_HYST_ASYM) {        // D3, Q14
    const float al = (fabsf(x) > fabsf(ha)) ? p.alpha_load : p.alpha_unload;
    h = fmaf(al, x - ha, ha);
    ha = h;
  }
  hrec = h;                                 // this step's signal, for the read-delay ring
  if (use_delayed) h = delayed;             // Eq. 25: y_{t - Delta_n}; bias, white noise and drift are those of step t
  drift = fmaf(p.sn_sigma_rw[cls], z_rw, drift);
  float y = fmaf(p.sn_sigma_white[cls], z_w, h + p.sn_bias[cls]) + drift;
  const float q = p.sn_quant[cls];
  if (q > 0.f) y = rintf(y / q) * q;        // quantize(., q): IEEE fp32 division, round half to even (R5)
  if (dead) y = fmaf(p.sn_stuck_max[cls] - p.sn_stuck_min[cls], stuck_u, p.sn_stuck_min[cls]);
  return y;
}

__device__ __forceinline__ float u24(uint32_t w) { return (float)(2u * (w >> 9) + 1u) * 5.9604644775390625e-8f; }

// Delta_n of the read delay (R9): max(0, Delta + k_n), k_n uniform on {-J..J}, ONE draw per (env, step) shared by every
// sensor of the env: stream 9, taxel word 0xffffffff (the draw the force / torque chain makes).
__device__ __forceinline__ int read_delay_steps(const TsStepParams& p, uint32_t env, uint32_t nstep, uint32_t ep4) {
  int delta = p.rd_delay;
  if (p.rd_jitter > 0) {
    const uint4 w = philox4x32_10(make_uint4(env, 0xffffffffu, nstep, ep4 | 9u), p.seed_lo, p.seed_hi);
    const int k = (int)(((unsigned long long)(w.x >> 9) * (unsigned long long)(2 * p.rd_jitter + 1)) >> 23) - p.rd_jitter;
    delta = max(0, p.rd_delay + k);
  }
  return delta;
}

// Threads [0, E T): depth + prox of one taxel (probe draws of the taxel: gain stream 3, dead flag from the state;
// stream 10 -> (z_rw, z_w) of depth and of prox, stream 11 -> stuck values).  Threads [E T, E T + E M): the three
// channels of one marker (probe 0x80000000 + m: streams 0 / 1 -> z_rw, z_w; 2 dead; 3 gain; 4 stuck).
template <int MODE>
__global__ void __launch_bounds__(256) ts_scalar_noise_kernel(const __grid_constant__ TsStepParams p) {
  const long long gt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long ET = (long long)p.E * p.T, EM = (long long)p.E * p.M;
  const bool gain_on = p.gain_min != 1.f || p.gain_max != 1.f;
  if (gt < ET) {
    if (!p.depth_noisy && !p.prox_noisy) return;
    const int e = (int)(gt / p.T), j = (int)(gt - (long long)e * p.T);
    const bool act = __ldg(&p.tx_pos[j].w) > 0.f;
    float od = 0.f, op = 0.f;
    if (act) {
      const uint32_t ep4 = __ldg(p.episode + e) << 4, env = p.env_id_base + (uint32_t)e;
      const uint32_t nstep = p.gstep - __ldg(p.reset_step + e);
      const uint4 w = philox4x32_10(make_uint4(env, (uint32_t)j, nstep, ep4 | 10u), p.seed_lo, p.seed_hi);
      float zd0, zd1, zp0, zp1;
      box_muller(w.x, w.y, zd0, zd1);
      box_muller(w.z, w.w, zp0, zp1);
      const bool dead = (p.st_flags[gt] >> 1) & 1;
      float gain = 1.f, su_d = 0.f, su_p = 0.f;
      if (gain_on) gain = fmaf(p.gain_max - p.gain_min, u24(philox4x32_10(make_uint4(env, (uint32_t)j, 0u, ep4 | 3u), p.seed_lo, p.seed_hi).x), p.gain_min);
      if (dead) {
        const uint4 ws = philox4x32_10(make_uint4(env, (uint32_t)j, 0u, ep4 | 11u), p.seed_lo, p.seed_hi);
        su_d = u24(ws.x); su_p = u24(ws.y);
      }
      float4 hs = MODE != TS_HYST_OFF ? p.sn_h[gt] : make_float4(0.f, 0.f, 0.f, 0.f);
      float2 dr = p.sn_d[gt];
      const float cd = p.depth_pert ? __ldcs(p.depth_pert + gt) : (p.depth ? p.depth[gt] : 0.f);
      const float cp = p.prox ? p.prox[gt] : 0.f;
      // read delay: ring slot n mod S holds the signal of step n (and of step n - S: read first, write last)
      const bool ring_on = p.sn_ring != nullptr && p.rd_S > 0;
      bool use_del = false;
      float2 del = make_float2(0.f, 0.f);
      float2* ring_w = nullptr;
      if (ring_on) {
        const unsigned S = (unsigned)p.rd_S;
        float2* const ring = p.sn_ring + (size_t)e * S * p.T + j;
        const int delta = read_delay_steps(p, env, nstep, ep4);
        use_del = delta > 0;
        if (use_del && nstep >= (uint32_t)delta) del = ring[(size_t)((nstep - (uint32_t)delta) % S) * p.T];   // else: before the episode (Q12)
        ring_w = ring + (size_t)(nstep % S) * p.T;
      }
      float2 rec = make_float2(0.f, 0.f);
      if (MODE == TS_HYST_MAXWELL) {
        od = scalar_chain<MODE>(p, 0, cd, gain, dead, su_d, zd0, zd1, hs.x, hs.y, dr.x, use_del, del.x, rec.x);
        op = scalar_chain<MODE>(p, 1, cp, gain, dead, su_p, zp0, zp1, hs.z, hs.w, dr.y, use_del, del.y, rec.y);
      } else {
        float dummy = 0.f;
        od = scalar_chain<MODE>(p, 0, cd, gain, dead, su_d, zd0, zd1, hs.x, dummy, dr.x, use_del, del.x, rec.x);
        op = scalar_chain<MODE>(p, 1, cp, gain, dead, su_p, zp0, zp1, hs.y, dummy, dr.y, use_del, del.y, rec.y);
      }
      if (ring_w) *ring_w = rec;
      if (MODE != TS_HYST_OFF) p.sn_h[gt] = hs;
      p.sn_d[gt] = dr;
    }
    if (p.depth_noisy) __stcs(p.depth_noisy + gt, od);
    if (p.prox_noisy) __stcs(p.prox_noisy + gt, op);
  } else if (gt < ET + EM) {
    if (!p.marker_noisy) return;
    const long long gm = gt - ET;
    const int e = (int)(gm / p.M), m = (int)(gm - (long long)e * p.M);
    // a marker is active iff its patch is (link filter): marker normals of filtered patches stay, radii go to 0
    const bool act = __ldg(&p.mk_pos[m].w) > 0.f;  // w = 1 for markers of active patches (set by ts_create)
    float out[3] = {0.f, 0.f, 0.f};
    if (act) {
      const uint32_t ep4 = __ldg(p.episode + e) << 4, env = p.env_id_base + (uint32_t)e, probe = 0x80000000u + (uint32_t)m;
      const uint32_t nstep = p.gstep - __ldg(p.reset_step + e);
      const uint4 w0 = philox4x32_10(make_uint4(env, probe, nstep, ep4 | 0u), p.seed_lo, p.seed_hi);
      const uint4 w1 = philox4x32_10(make_uint4(env, probe, nstep, ep4 | 1u), p.seed_lo, p.seed_hi);
      float zr[4], zw[2];
      box_muller(w0.x, w0.y, zr[0], zr[1]);
      box_muller(w0.z, w0.w, zr[2], zr[3]);
      box_muller(w1.x, w1.y, zw[0], zw[1]);
      const bool dead = philox4x32_10(make_uint4(env, probe, 0u, ep4 | 2u), p.seed_lo, p.seed_hi).x < p.dead_thr;
      float gain = 1.f;
      if (gain_on) gain = fmaf(p.gain_max - p.gain_min, u24(philox4x32_10(make_uint4(env, probe, 0u, ep4 | 3u), p.seed_lo, p.seed_hi).x), p.gain_min);
      uint4 ws = make_uint4(0u, 0u, 0u, 0u);
      if (dead) ws = philox4x32_10(make_uint4(env, probe, 0u, ep4 | 4u), p.seed_lo, p.seed_hi);
      const uint32_t wsv[3] = {ws.x, ws.y, ws.z};
      float* hp = p.sm_h + gm * 6;
      float* dp = p.sm_d + gm * 3;
      const float* cm = p.marker + gm * 3;
      const bool ring_on = p.sm_ring != nullptr && p.rd_S > 0;
      bool use_del = false;
      float del[3] = {0.f, 0.f, 0.f};
      float* ring_w = nullptr;
      if (ring_on) {
        const unsigned S = (unsigned)p.rd_S;
        float* const ring = p.sm_ring + ((size_t)e * S * p.M + m) * 3;
        const int delta = read_delay_steps(p, env, nstep, ep4);
        use_del = delta > 0;
        if (use_del && nstep >= (uint32_t)delta) {
          const float* r = ring + (size_t)((nstep - (uint32_t)delta) % S) * p.M * 3;
          del[0] = r[0]; del[1] = r[1]; del[2] = r[2];
        }
        ring_w = ring + (size_t)(nstep % S) * p.M * 3;
      }
      float rec[3];
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        float ha = MODE != TS_HYST_OFF ? hp[c] : 0.f, hb = MODE == TS_HYST_MAXWELL ? hp[3 + c] : 0.f, dr = dp[c];
        out[c] = scalar_chain<MODE>(p, 2, cm[c], gain, dead, u24(wsv[c]), zr[c], c == 0 ? zr[3] : zw[c - 1], ha, hb, dr, use_del,
                                    del[c], rec[c]);
        if (MODE != TS_HYST_OFF) hp[c] = ha;
        if (MODE == TS_HYST_MAXWELL) hp[3 + c] = hb;
        dp[c] = dr;
      }
      if (ring_w) { ring_w[0] = rec[0]; ring_w[1] = rec[1]; ring_w[2] = rec[2]; }
    }
    float* o = p.marker_noisy + gm * 3;
    __stcs(o, out[0]); __stcs(o + 1, out[1]); __stcs(o + 2, out[2]);
  }
}

// zeroes the state of the noisy scalar readouts for the masked envs
__global__ void ts_reset_scalar_kernel(const __grid_constant__ TsStepParams p, const uint8_t* mask) {
  const long long gt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int per = p.T > p.M ? p.T : p.M;
  if (gt >= (long long)p.E * per) return;
  const int e = (int)(gt / per), i = (int)(gt - (long long)e * per);
  if (mask && !mask[e]) return;
  if (i < p.T && p.sn_d) {
    p.sn_h[(size_t)e * p.T + i] = make_float4(0.f, 0.f, 0.f, 0.f);
    p.sn_d[(size_t)e * p.T + i] = make_float2(0.f, 0.f);
  }
  if (i < p.M && p.sm_d) {
    for (int c = 0; c < 6; ++c) p.sm_h[((size_t)e * p.M + i) * 6 + c] = 0.f;
    for (int c = 0; c < 3; ++c) p.sm_d[((size_t)e * p.M + i) * 3 + c] = 0.f;
  }
}

// ---------------------------------------------------------------------------------------
// App. A.6 point-cloud ProximityTaxel (Eq. 12-17).  One thread per (env, taxel).
// The tracked points are static in their object's frame, so each cloud was sorted once into a uniform grid of cell
// size R_j / TS_PC_REACH (ts_set_pointclouds): the taxel centre is taken into the object frame (double), the rows of
// cells that reach into its sensing sphere are scanned, and of the points inside the sensing sphere only two sums are kept,
//     S0 = sum_i P_ij,   S1 = sum_i P_ij (p_i - q_j)          (P_ij = R_j - |p_i - q_j|, Eq. 12)
// because Eq. 13-17 are linear in p_i:  v_p,i - v_tax = A + w_O x (p_i - q_j),  A = v_O + w_O x (q_j - p_O) - v_tax, so
//     sum_i P_ij v_t,ij = Pi_a (S0 A + w_O x S1),   f^w = k rho S0 a + k_s rho Pi_a(...),   tau^w = k rho S1 x a.
// Same result as the per-point sums of the paper up to rounding order.  Distances and the two sums in fp32 on fp32
// differences of nearby points (a few hundred terms of bounded size: ~1e-6 relative), the rest in double.
// ---------------------------------------------------------------------------------------
#ifndef TS_PC_GROUP
#define TS_PC_GROUP 4   // lanes that scan one taxel's neighbourhood together (32 / TS_PC_GROUP taxels per warp round)
#endif
// The scan is bound by the latency of its dependent loads (run bounds -> points), so residency matters more than
// registers: 12 blocks of 128 threads per SM (40 registers; the double-precision pose data that lives across the scan is
// spilled around it) runs 1.40 ms where 4 blocks (128 registers, nothing spilled) run 2.62 ms (config-4 scene, 4,096 envs).
#ifndef TS_PC_MINB
#define TS_PC_MINB 12
#endif
__global__ void __launch_bounds__(128, TS_PC_MINB) ts_proxpc_kernel(const __grid_constant__ TsStepParams p) {
  // Thread = (env, taxel) for the pose arithmetic and the force / torque; the SCAN of a taxel's neighbourhood is shared
  // by TS_PC_GROUP lanes: a thread-per-taxel scan runs every warp to its longest neighbourhood at ~14 of 32 lanes (ncu),
  // the shared scan keeps the lanes busy and splits each run of points.  Every lane of the warp stays in the kernel
  // (shuffles below): threads past the end and filler taxels carry ok = false.
  const long long gt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const bool in_range = gt < (long long)p.E * p.T;
  const int lane = threadIdx.x & 31;
  const int e = in_range ? (int)(gt / p.T) : 0, j = in_range ? (int)(gt - (long long)e * p.T) : 0;
  const float4 P4 = __ldg(p.tx_pos + j);
  const bool act = in_range && P4.w > 0.f;
  float out[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  double RL[9];
  D3 pL = D3{0.0, 0.0, 0.0}, q = pL, a = pL, vtax = pL;
  double rho = 0.0;
  if (act) {
    const int pidx = __ldg(p.tx_patch + j);
    const TsPatch& pt = p.patches[pidx];
    const int link = __ldg(&pt.link);
    const float4 na = __ldg(&pt.na);
    const size_t el = (size_t)e * p.L + link;
    quat_Rd(p.link_quat + el * 4, RL);
    pL = ld3d(p.link_pos + el * 3);
    q = pL + mulR(RL, D3{(double)P4.x, (double)P4.y, (double)P4.z});       // Eq. 1
    a = mulR(RL, D3{(double)na.x, (double)na.y, (double)na.z});
    vtax = ld3d(p.link_linvel + el * 3) + cross(ld3d(p.link_angvel + el * 3), q - pL);   // Eq. 13
    long long n_track = 0;
    for (int k = 0; k < p.K; ++k) n_track += __ldg(p.pc_id + (size_t)e * p.K + k) >= 0 ? p.pc_n : 0;
    rho = (double)p.pc_density / (double)(n_track > 0 ? n_track : 1);          // Eq. 15 (Q27)
  }
  const float R = p.pc_radius, R2 = R * R;
  D3 fw = D3{0.0, 0.0, 0.0}, tw = D3{0.0, 0.0, 0.0};
  for (int k = 0; k < p.K; ++k) {   // warp-uniform
    const size_t ek = (size_t)e * p.K + k;
    const int id = act ? __ldg(p.pc_id + ek) : -1;
    double RO[9];
    D3 pO = D3{0.0, 0.0, 0.0};
    float xf = 0.f, yf = 0.f, zf = 0.f;
    if (id >= 0) {
      quat_Rd(p.obj_quat + ek * 4, RO);
      pO = ld3d(p.obj_pos + ek * 3);
      const D3 xd = mulRT(RO, q - pO);                                                       // taxel centre, object frame
      xf = (float)xd.x; yf = (float)xd.y; zf = (float)xd.z;
    }
    // ---- shared scan: in round r the TS_PC_GROUP lanes of group gq serve the taxel of lane r * NG + gq
    constexpr int NG = 32 / TS_PC_GROUP;          // groups per warp = taxels per round
    const int gq = lane / TS_PC_GROUP, sub = lane % TS_PC_GROUP;
    float S0f = 0.f, S1xf = 0.f, S1yf = 0.f, S1zf = 0.f;   // this lane's own taxel: filled in its round
    if (__any_sync(TS_FULL, id >= 0)) {
#pragma unroll 1
      for (int r = 0; r < TS_PC_GROUP; ++r) {
        const int owner = r * NG + gq;
        const int oid = __shfl_sync(TS_FULL, id, owner);
        const float ox = __shfl_sync(TS_FULL, xf, owner), oy = __shfl_sync(TS_FULL, yf, owner), oz = __shfl_sync(TS_FULL, zf, owner);
        float s0 = 0.f, sx = 0.f, sy = 0.f, sz = 0.f;
        if (oid >= 0) {
          const TsPcGrid g = p.pc_grid[oid];
          const int ci = (int)floorf((ox - g.ox) * g.inv_cell), cj = (int)floorf((oy - g.oy) * g.inv_cell), ck = (int)floorf((oz - g.oz) * g.inv_cell);
          const float cellw = 1.0f / g.inv_cell;
          const float ry = oy - g.oy, rz = oz - g.oz;       // position relative to the grid origin
          const int i0 = max(ci - TS_PC_REACH, 0), i1 = min(ci + TS_PC_REACH, g.nx - 1);
          const float4* pts = p.pc_pts + g.pt0;
          if (i0 <= i1) {
            for (int dk = -TS_PC_REACH; dk <= TS_PC_REACH; ++dk) {
              const int kk = ck + dk;
              if (kk < 0 || kk >= g.nz) continue;
              const float gz = fmaxf(fmaxf((float)kk * cellw - rz, rz - (float)(kk + 1) * cellw), 0.f);   // gap to the slab in z
              for (int dj = -TS_PC_REACH; dj <= TS_PC_REACH; ++dj) {
                const int jj = cj + dj;
                if (jj < 0 || jj >= g.ny) continue;
                const float gy = fmaxf(fmaxf((float)jj * cellw - ry, ry - (float)(jj + 1) * cellw), 0.f);
                // the whole row of cells lies outside the sensing sphere (1e-6 m of slack for the rounding of the cell edges)
                if (fmaf(gy, gy, gz * gz) >= (R + 1e-6f) * (R + 1e-6f)) continue;
                // the x-neighbours of a row are consecutive cells: one contiguous run of points, split over the group's lanes
                const int row = g.cell0 + (kk * g.ny + jj) * g.nx;
                const int b = __ldg(p.pc_cell + row + i0), en = __ldg(p.pc_cell + row + i1 + 1);
                for (int i = b + sub; i < en; i += TS_PC_GROUP) {
                  const float4 pp = __ldg(pts + i);
                  const float dx = pp.x - ox, dy = pp.y - oy, dz = pp.z - oz;
                  const float d2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                  const float P = d2 < R2 ? R - sqrtf(d2) : 0.f;                             // Eq. 12 (0 outside the sphere)
                  s0 += P;
                  sx = fmaf(P, dx, sx); sy = fmaf(P, dy, sy); sz = fmaf(P, dz, sz);
                }
              }
            }
          }
        }
        // sum over the group's lanes (fp32: <= a few hundred terms of bounded size), then hand the totals to the owner
#pragma unroll
        for (int o = TS_PC_GROUP / 2; o > 0; o >>= 1) {
          s0 += __shfl_xor_sync(TS_FULL, s0, o); sx += __shfl_xor_sync(TS_FULL, sx, o);
          sy += __shfl_xor_sync(TS_FULL, sy, o); sz += __shfl_xor_sync(TS_FULL, sz, o);
        }
        const int src = (lane % NG) * TS_PC_GROUP;      // first lane of the group that served THIS lane's taxel in round lane / NG
        const float t0 = __shfl_sync(TS_FULL, s0, src), tx = __shfl_sync(TS_FULL, sx, src), ty = __shfl_sync(TS_FULL, sy, src),
                    tz = __shfl_sync(TS_FULL, sz, src);
        if (lane / NG == r) { S0f = t0; S1xf = tx; S1yf = ty; S1zf = tz; }
      }
    }
    if (id >= 0 && S0f > 0.f) {
      const double S0 = (double)S0f;
      const D3 S1w = mulR(RO, D3{(double)S1xf, (double)S1yf, (double)S1zf});                 // sum P (p_i - q_j), world axes
      const D3 wO = ld3d(p.obj_angvel + ek * 3);
      const D3 A = ld3d(p.obj_linvel + ek * 3) + cross(wO, q - pO) - vtax;                   // Eq. 13 at p_i = q_j
      const D3 sv = S0 * A + cross(wO, S1w);                                                 // sum P (v_p - v_tax)
      const D3 st = sv - dot(sv, a) * a;                                                     // Eq. 14 (linear)
      fw = fw + ((double)p.pc_k * rho * S0) * a + ((double)p.pc_ks * rho) * st;              // Eq. 16
      tw = tw + ((double)p.pc_k * rho) * cross(S1w, a);                                      // Eq. 17
    }
  }
  if (act) {
    const D3 fl = mulRT(RL, fw), tl = mulRT(RL, tw);                                         // reported in the link frame
    out[0] = (float)fl.x; out[1] = (float)fl.y; out[2] = (float)fl.z; out[3] = (float)tl.x; out[4] = (float)tl.y; out[5] = (float)tl.z;
  }
  if (in_range) store6(p.proxpc + gt * 6, out);
}

// ---------------------------------------------------------------------------------------
// App. A.7 elastomer shear history (Eq. 22-23; reading R11).  One block per (env, patch with markers).
// Phase A: the relative pose link <- object in double (z_p = t + Rm p^o, sensor-link frame).
// Phase B: every thread walks tracked points: pad SDF phi_el = n . (z_p - x_c) over the pad, anchor update
//          (set below -eta_enter, cleared above +eta_exit; decisions in double like the oracle), and the anchored,
//          penetrating points (a few tens per touching pad) are queued in shared memory.
// Phase C: one thread per marker sums s_s Pi_n(z_p - e_p) h_p exp(-lambda_s |Pi_n(x_j - z_p)|^2) over the queue and adds
//          it to the dilation value the step kernel wrote (Eq. 23).
// ---------------------------------------------------------------------------------------
#define TS_SHEAR_Q 512
// 2 / 4 / 6 / 8 blocks per SM: 1.38 / 0.84 / 0.68 / 0.73 ms (the point loop waits on its loads).
#ifndef TS_SH_MINB
#define TS_SH_MINB 6
#endif
__global__ void __launch_bounds__(256, TS_SH_MINB) ts_shear_kernel(const __grid_constant__ TsStepParams p) {
  __shared__ double Rm[9], tv[3];
  __shared__ float prism[12];         // the pad's frame in the object frame: u = a_u . p + b_u, v = a_v . p + b_v, phi_el = a_n . p + b_n
  __shared__ int b2_on, dcnt;         // can any point of the cloud lie behind the pad plane?  change of the anchored count
  __shared__ float4 qd[TS_SHEAR_Q];   // (tangential slide x, y, z, h_p)
  __shared__ float4 qz[TS_SHEAR_Q];   // z_p relative to the pad centre
  __shared__ int wcnt[2][8];          // queued points per warp of the current pass (double-buffered by pass parity)
  __shared__ uint4 fl[256];           // anchor flags of the current chunk, 16 per thread
  __shared__ int pfx[257];            // exclusive prefix of the set flags per thread; [256] = total
  __shared__ int wtot[8];
  // Blocks run in the step kernel's env order: the relative poses of this step are still in frames_g (row bx = env
  // env_perm[bx]), so no pose is rebuilt here (a one-thread rebuild was most of a block's life for pads that touch nothing).
  const int bx = blockIdx.x / p.P, pi = blockIdx.x - bx * p.P, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int e = p.env_perm ? __ldg(p.env_perm + bx) : bx;
  const TsPatch& pt = p.patches[pi];
  const int mcount = __ldg(&pt.mnu) * __ldg(&pt.mnv), link = __ldg(&pt.link);
  if (mcount == 0 || link < 0) return;
  if (!(__ldg(&p.tx_pos[__ldg(&pt.start)].w) > 0.f)) return;       // link filtered out: fillers
  const float4 na = __ldg(&pt.na), ua = __ldg(&pt.ua), va = __ldg(&pt.va), ctr = __ldg(&pt.ctr);
  const D3 n = D3{(double)na.x, (double)na.y, (double)na.z}, uu = D3{(double)ua.x, (double)ua.y, (double)ua.z}, vv = D3{(double)va.x, (double)va.y, (double)va.z};
  const D3 xc = D3{(double)ctr.x, (double)ctr.y, (double)ctr.z};
  const double hu = 0.5 * (double)ua.w, hv = 0.5 * (double)va.w;
  const int N = p.pc_n, Np = p.pc_np;
  float ax = 0.f, ay = 0.f, az = 0.f;   // this thread's marker (tid < mcount): shear sum
  float mx = 0.f, my = 0.f, mz = 0.f;
  if (tid < mcount) {
    const float4 mp = __ldg(p.mk_pos + __ldg(&pt.mstart) + tid);
    mx = mp.x - ctr.x; my = mp.y - ctr.y; mz = mp.z - ctr.z;
  }
  int qn = 0;                            // queue fill: the same value in every thread (block-uniform)
  auto shear_drain = [&]() {             // phase C over the queued points (call between barriers)
    if (tid >= mcount) return;
    for (int s2 = 0; s2 < qn; ++s2) {
      const float4 d4 = qd[s2], z4 = qz[s2];
      const float rx = mx - z4.x, ry = my - z4.y, rz = mz - z4.z;
      const float rn = fmaf(rx, na.x, fmaf(ry, na.y, rz * na.z));
      const float tx = fmaf(-rn, na.x, rx), ty = fmaf(-rn, na.y, ry), tz = fmaf(-rn, na.z, rz);   // Pi_n(x_j - z_p)
      const float wgt = p.s_s * d4.w * expf(-p.lambda_s * fmaf(tx, tx, fmaf(ty, ty, tz * tz)));   // Eq. 22
      ax = fmaf(wgt, d4.x, ax); ay = fmaf(wgt, d4.y, ay); az = fmaf(wgt, d4.z, az);
    }
  };
  // pad SDF of a tracked point given in the object frame (R11): +inf beside the pad, n . (z - x_c) over it
  auto pad_phi = [&](float4 po, D3& rel) {
    const D3 z = D3{tv[0], tv[1], tv[2]} + mulR(Rm, D3{(double)po.x, (double)po.y, (double)po.z});
    rel = z - xc;
    double phi_el = __longlong_as_double(0x7ff0000000000000LL);
    if (fabs(dot(rel, uu)) <= hu && fabs(dot(rel, vv)) <= hv) phi_el = dot(rel, n);
    return phi_el;
  };
  int pass = 0;
  for (int k = 0; k < p.K; ++k) {
    const int id = __ldg(p.pc_id + (size_t)e * p.K + k);   // block-uniform
    if (id < 0) continue;
    __syncthreads();
    if (tid < 12) {   // R_L^T R_O = M^T and R_L^T (p_O - p_L) = -cbar of the frame (link of this pad, object k)
      const FrameS* F = reinterpret_cast<const FrameS*>(p.frames_g) + ((size_t)bx * p.P + pi) * p.K + k;
      if (tid < 9) Rm[tid] = F->M[(tid % 3) * 3 + tid / 3];
      else tv[tid - 9] = -F->cbar[tid - 9];
    }
    __syncthreads();
    if (tid == 0) {
      const D3 t = D3{tv[0], tv[1], tv[2]};
      const D3 au = mulRT(Rm, uu), av = mulRT(Rm, vv), tc = t - xc;
      prism[0] = (float)au.x; prism[1] = (float)au.y; prism[2] = (float)au.z; prism[3] = (float)dot(uu, tc);
      prism[4] = (float)av.x; prism[5] = (float)av.y; prism[6] = (float)av.z; prism[7] = (float)dot(vv, tc);
      const D3 an = mulRT(Rm, n);
      const double bn = dot(n, tc);
      prism[8] = (float)an.x; prism[9] = (float)an.y; prism[10] = (float)an.z; prism[11] = (float)bn;
      // smallest phi_el over the cloud's bounding box: if even that is not behind the pad plane, nothing can anchor
      const TsPcGrid g = p.pc_grid[id];
      const double w = 1.0 / (double)g.inv_cell;
      const double lo3[3] = {(double)g.ox, (double)g.oy, (double)g.oz}, ext[3] = {g.nx * w, g.ny * w, g.nz * w}, a3[3] = {an.x, an.y, an.z};
      double pmin = bn;
      for (int ax2 = 0; ax2 < 3; ++ax2) pmin += fmin(a3[ax2] * lo3[ax2], a3[ax2] * (lo3[ax2] + ext[ax2]));
      b2_on = pmin < -(double)p.eta_enter + 1e-6 ? 1 : 0;
      dcnt = 0;
    }
    __syncthreads();
    const size_t sbase = (((size_t)e * p.P + pi) * p.K + k) * (size_t)Np;   // a multiple of 16: the flag rows are 16-byte aligned
    int* const cntp = p.sh_cnt + ((size_t)e * p.P + pi) * p.K + k;          // anchored points of this (env, pad, object)
    const int cnt0 = *cntp;                                                  // block-uniform
    const int NpB1 = cnt0 > 0 ? Np : 0;                                      // nothing anchored: no flag scan at all
    // ---- phase B1: the points that are anchored, found by a scan of the flag bytes (16 per thread and chunk), taken in
    // index order: exit test, and the penetrating ones go to the queue.  Work ~ N / 16 loads + the anchored points.
    for (int c0 = 0; c0 < NpB1; c0 += 4096) {
      __syncthreads();                     // fl / pfx of the previous chunk are no longer read
      uint4 f = make_uint4(0u, 0u, 0u, 0u);
      const int off = c0 + tid * 16;
      if (off < Np) f = *reinterpret_cast<const uint4*>(p.sh_on + sbase + off);
      fl[tid] = f;
      const int cnt = __popc(f.x & 0x01010101u) + __popc(f.y & 0x01010101u) + __popc(f.z & 0x01010101u) + __popc(f.w & 0x01010101u);
      int inc = cnt;                       // inclusive scan inside the warp
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(TS_FULL, inc, o);
        if (lane >= o) inc += v;
      }
      if (lane == 31) wtot[warp] = inc;
      __syncthreads();
      int wb = 0, total = 0;
#pragma unroll
      for (int w2 = 0; w2 < 8; ++w2) {
        const int c2 = wtot[w2];
        if (w2 < warp) wb += c2;
        total += c2;
      }
      pfx[tid] = wb + inc - cnt;
      if (tid == 0) pfx[256] = total;
      __syncthreads();
      for (int m0 = 0; m0 < total; m0 += 256, ++pass) {
        if (qn > TS_SHEAR_Q - 256) {       // a pass queues at most 256 points: drain before the queue could overflow
          __syncthreads();
          shear_drain();
          qn = 0;
          __syncthreads();
        }
        const int m = m0 + tid;
        bool push = false;
        float4 vd = make_float4(0.f, 0.f, 0.f, 0.f), vz = vd;
        if (m < total) {
          int lo = 0, hi = 255;            // owner: the last thread whose prefix is <= m
          while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (pfx[mid] <= m) lo = mid; else hi = mid - 1;
          }
          const uint4 g = fl[lo];
          const unsigned wv[4] = {g.x, g.y, g.z, g.w};
          int kth = m - pfx[lo], byte = 0;
#pragma unroll
          for (int b2 = 0; b2 < 16; ++b2) {
            const int bit = (int)((wv[b2 >> 2] >> ((b2 & 3) * 8)) & 1u);
            if (bit && kth == 0) byte = b2;
            kth -= bit;
          }
          const int i = c0 + lo * 16 + byte;   // < N: flags past N are never set
          D3 rel;
          const double phi_el = pad_phi(__ldg(p.pc_raw + (size_t)id * N + i), rel);
          if (phi_el > (double)p.eta_exit) {
            p.sh_on[sbase + i] = 0;
            atomicSub(&dcnt, 1);
          } else if (phi_el < 0.0) {
            const float4 anc = p.sh_e[sbase + i];
            const D3 dz = D3{rel.x - (double)anc.x, rel.y - (double)anc.y, rel.z - (double)anc.z};
            const D3 dzt = dz - dot(dz, n) * n;                          // Pi_n(z_p - e_p)
            push = true;
            vd = make_float4((float)dzt.x, (float)dzt.y, (float)dzt.z, (float)(-phi_el));
            vz = make_float4((float)rel.x, (float)rel.y, (float)rel.z, 0.f);
          }
        }
        // Ordered compaction: the queue holds the anchored points in index order, so the fp32 sums below are the same
        // from run to run (a shared-memory atomic counter would enqueue in arrival order).
        const unsigned bal = __ballot_sync(TS_FULL, push);
        if (lane == 0) wcnt[pass & 1][warp] = __popc(bal);
        __syncthreads();
        int base = qn, tot = 0;
#pragma unroll
        for (int w2 = 0; w2 < 8; ++w2) {
          const int c2 = wcnt[pass & 1][w2];
          if (w2 < warp) base += c2;
          tot += c2;
        }
        if (push) {
          const int slot = base + __popc(bal & ((1u << lane) - 1u));     // < TS_SHEAR_Q by the drain rule above
          qd[slot] = vd; qz[slot] = vz;
        }
        qn += tot;
      }
    }
    __syncthreads();
    shear_drain();
    qn = 0;
    // ---- phase B2: new anchors.  Only points inside the pad's prism can anchor, so the cloud's grid is walked by rows
    // of cells (x fastest): per row the x-interval that can meet the prism, then the points of that run of cells that are
    // not anchored yet.  A point anchored here contributes nothing this step (z_p = e_p), so it is not queued.
    if (b2_on) {   // block-uniform
      const TsPcGrid g = p.pc_grid[id];
      const float cw = __frcp_rn(g.inv_cell), rc = 0.7072f * cw + 1e-5f;
      const float Hu = (float)hu + rc, Hv = (float)hv + rc, Hn = rc - p.eta_enter;
      const float4* pts = p.pc_pts + g.pt0;
      const int nrows = g.ny * g.nz;
      const float inv_ny = 1.0f / (float)g.ny;
      int* const runb = reinterpret_cast<int*>(fl);   // first point of each thread's run (fl is free after phase B1)
      for (int r0 = 0; r0 < nrows; r0 += 256) {
        // one row of cells per thread: the run of points that can meet the prism behind the pad plane (possibly empty)
        const int row = r0 + tid;
        int rb = 0, rlen = 0;
        if (row < nrows) {
          const int kk = (int)(((float)row + 0.5f) * inv_ny), jj = row - kk * g.ny;   // exact: row, ny < 2^20
          const float yc = g.oy + ((float)jj + 0.5f) * cw, zc = g.oz + ((float)kk + 0.5f) * cw;
          float xlo = g.ox, xhi = g.ox + (float)g.nx * cw;
          bool any = true;
#pragma unroll
          for (int s2 = 0; s2 < 3; ++s2) {   // slabs |u| <= Hu, |v| <= Hv and the half-space phi_el <= Hn along the line (x, yc, zc)
            const float a = prism[4 * s2], c1 = fmaf(prism[4 * s2 + 1], yc, fmaf(prism[4 * s2 + 2], zc, prism[4 * s2 + 3]));
            const float H = s2 == 0 ? Hu : (s2 == 1 ? Hv : Hn);
            if (fabsf(a) < 1e-6f) {
              any = any && c1 <= H + 1e-4f && (s2 == 2 || c1 >= -H - 1e-4f);
            } else {
              const float ia = __frcp_rn(a);
              const float x1 = (H - c1) * ia, x0 = s2 == 2 ? (a > 0.f ? -3.0e38f : 3.0e38f) : (-H - c1) * ia;
              xlo = fmaxf(xlo, fminf(x0, x1)); xhi = fminf(xhi, fmaxf(x0, x1));
            }
          }
          if (any && xlo <= xhi) {           // +- one cell of slack covers the rounding of the interval ends
            const int i0 = max((int)floorf((xlo - g.ox) * g.inv_cell) - 1, 0), i1 = min((int)floorf((xhi - g.ox) * g.inv_cell) + 1, g.nx - 1);
            if (i0 <= i1) {
              const int cell = g.cell0 + row * g.nx;
              rb = __ldg(p.pc_cell + cell + i0);
              rlen = __ldg(p.pc_cell + cell + i1 + 1) - rb;
            }
          }
        }
        // the candidates of all rows, dealt to the threads one point each (a row's thread walking its own run left 3 of 32
        // lanes busy): block prefix of the run lengths, then point m belongs to the last row whose prefix is <= m
        __syncthreads();                     // runb / pfx of the previous batch (or of phase B1) are no longer read
        runb[tid] = rb;
        int inc = rlen;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const int v = __shfl_up_sync(TS_FULL, inc, o);
          if (lane >= o) inc += v;
        }
        if (lane == 31) wtot[warp] = inc;
        __syncthreads();
        int wb = 0, total = 0;
#pragma unroll
        for (int w2 = 0; w2 < 8; ++w2) {
          const int c2 = wtot[w2];
          if (w2 < warp) wb += c2;
          total += c2;
        }
        pfx[tid] = wb + inc - rlen;
        __syncthreads();
        for (int m = tid; m < total; m += 256) {
          int lo = 0, hi = 255;
          while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (pfx[mid] <= m) lo = mid; else hi = mid - 1;
          }
          const float4 po = __ldg(pts + runb[lo] + (m - pfx[lo]));
          const int i = __float_as_int(po.w);                            // index of the point in the caller's order
          if (p.sh_on[sbase + i]) continue;
          D3 rel;
          const double phi_el = pad_phi(po, rel);
          if (phi_el < -(double)p.eta_enter) {
            p.sh_on[sbase + i] = 1;
            p.sh_e[sbase + i] = make_float4((float)rel.x, (float)rel.y, (float)rel.z, 0.f);
            atomicAdd(&dcnt, 1);
          }
        }
      }
    }
    __syncthreads();
    if (tid == 0 && dcnt != 0) *cntp = cnt0 + dcnt;
  }
  if (tid < mcount && (ax != 0.f || ay != 0.f || az != 0.f)) {
    float* o = p.marker + ((size_t)e * p.M + __ldg(&pt.mstart) + tid) * 3;
    o[0] += ax; o[1] += ay; o[2] += az;                               // Eq. 23
  }
}

__global__ void ts_reset_shear_kernel(const __grid_constant__ TsStepParams p, const uint8_t* mask) {
  const size_t per = (size_t)p.P * p.K * p.pc_np;
  const size_t gt = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (gt >= (size_t)p.E * per) return;
  const int e = (int)(gt / per);
  if (mask && !mask[e]) return;
  p.sh_on[gt] = 0;
  const size_t r = gt - (size_t)e * per;
  if (r < (size_t)p.P * p.K) p.sh_cnt[(size_t)e * p.P * p.K + r] = 0;   // anchored-point counters of the env
}

// ---------------------------------------------------------------------------------------
// App. A.1 raycast contact-depth backend (reading Q28).  One thread per (env, taxel): the probe centre and
// normal go into the object frame (double), the mesh's bounding volume hierarchy is walked with a private stack
// (a node is entered when its box meets the probe sphere; the ray segment of length R_j lies inside that sphere), and
// every triangle of a reached leaf takes the sphere-triangle closest-point test (penetration R_j - dist) and the
// ray-triangle test from the centre along -a_j (penetration R_j - hit distance).  The deepest wins; its face normal
// is reported in the sensor-link frame.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ F3 sub3(F3 a, F3 b) { return mk3(a.x - b.x, a.y - b.y, a.z - b.z); }
__device__ __forceinline__ F3 cross3(F3 a, F3 b) { return mk3(a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x); }

// closest point of triangle (a, b, c) to p (Voronoi-region walk; Ericson 5.1.5 restated in fp32)
__device__ __forceinline__ F3 closest_pt_tri(F3 p, F3 a, F3 b, F3 c) {
  const F3 ab = sub3(b, a), ac = sub3(c, a), ap = sub3(p, a);
  const float d1 = dot(ab, ap), d2 = dot(ac, ap);
  if (d1 <= 0.f && d2 <= 0.f) return a;
  const F3 bp = sub3(p, b);
  const float d3 = dot(ab, bp), d4 = dot(ac, bp);
  if (d3 >= 0.f && d4 <= d3) return b;
  const float vc = d1 * d4 - d3 * d2;
  if (vc <= 0.f && d1 >= 0.f && d3 <= 0.f) return a + (d1 / (d1 - d3)) * ab;
  const F3 cp = sub3(p, c);
  const float d5 = dot(ab, cp), d6 = dot(ac, cp);
  if (d6 >= 0.f && d5 <= d6) return c;
  const float vb = d5 * d2 - d1 * d6;
  if (vb <= 0.f && d2 >= 0.f && d6 <= 0.f) return a + (d2 / (d2 - d6)) * ac;
  const float va = d3 * d6 - d5 * d4;
  if (va <= 0.f && (d4 - d3) >= 0.f && (d5 - d6) >= 0.f) return b + ((d4 - d3) / ((d4 - d3) + (d5 - d6))) * sub3(c, b);
  const float den = 1.f / (va + vb + vc);
  return a + (vb * den) * ab + (vc * den) * ac;
}

// ray (o, unit d) against (a, b, c), both faces (Moeller-Trumbore restated): hit distance >= 0 or -1
__device__ __forceinline__ float ray_tri(F3 o, F3 d, F3 a, F3 b, F3 c) {
  const F3 e1 = sub3(b, a), e2 = sub3(c, a), pv = cross3(d, e2);
  const float det = dot(e1, pv);
  if (fabsf(det) < 1e-30f) return -1.f;
  const float inv = 1.f / det;
  const F3 tv = sub3(o, a);
  const float u = dot(tv, pv) * inv;
  if (u < 0.f || u > 1.f) return -1.f;
  const F3 qv = cross3(tv, e1);
  const float v = dot(d, qv) * inv;
  if (v < 0.f || u + v > 1.f) return -1.f;
  const float t = dot(e2, qv) * inv;
  return t >= 0.f ? t : -1.f;
}

// Latency-bound tree walk: residency beats registers (4 / 8 / 12 / 16 blocks per SM: 1.35 / 0.85 / 0.80 / 0.90 ms).
#ifndef TS_RC_MINB
#define TS_RC_MINB 12
#endif
__global__ void __launch_bounds__(128, TS_RC_MINB) ts_raycast_kernel(const __grid_constant__ TsStepParams p) {
  const long long gt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gt >= (long long)p.E * p.T) return;
  const int e = (int)(gt / p.T), j = (int)(gt - (long long)e * p.T);
  const float4 P4 = __ldg(p.tx_pos + j);
  float best = 0.f;
  D3 bn = D3{0.0, 0.0, 0.0};
  if (P4.w > 0.f) {
    const TsPatch& pt = p.patches[__ldg(p.tx_patch + j)];
    const int link = __ldg(&pt.link);
    const float4 na = __ldg(&pt.na);
    const size_t el = (size_t)e * p.L + link;
    double RL[9];
    quat_Rd(p.link_quat + el * 4, RL);
    const D3 q = ld3d(p.link_pos + el * 3) + mulR(RL, D3{(double)P4.x, (double)P4.y, (double)P4.z});   // Eq. 1
    const D3 a = mulR(RL, D3{(double)na.x, (double)na.y, (double)na.z});
    const float R = P4.w, R2 = R * R;
    for (int k = 0; k < p.K; ++k) {
      const int id = __ldg(p.rc_id + (size_t)e * p.K + k);
      if (id < 0) continue;
      const size_t ek = (size_t)e * p.K + k;
      double RO[9];
      quat_Rd(p.obj_quat + ek * 4, RO);
      const D3 qd = mulRT(RO, q - ld3d(p.obj_pos + ek * 3)), ad = mulRT(RO, a);
      const F3 qo = mk3((float)qd.x, (float)qd.y, (float)qd.z), nd = mk3(-(float)ad.x, -(float)ad.y, -(float)ad.z);
      int stack[48];
      int sp = 0;
      stack[sp++] = __ldg(p.rc_root + id);
      F3 wn = mk3(0.f, 0.f, 0.f);
      bool won = false;
      while (sp > 0) {
        const int node = stack[--sp];
        const float4 n0 = __ldg(p.rc_nodes + 2 * node), n1 = __ldg(p.rc_nodes + 2 * node + 1);
        const float dx = fmaxf(fmaxf(n0.x - qo.x, qo.x - n1.x), 0.f), dy = fmaxf(fmaxf(n0.y - qo.y, qo.y - n1.y), 0.f),
                    dz = fmaxf(fmaxf(n0.z - qo.z, qo.z - n1.z), 0.f);
        if (fmaf(dx, dx, fmaf(dy, dy, dz * dz)) >= R2) continue;           // the box misses the probe sphere
        const int cnt = __float_as_int(n1.w);
        if (cnt > 0) {
          const int first = __float_as_int(n0.w);
          for (int f = first; f < first + cnt; ++f) {
            const float4 A4 = __ldg(p.rc_tri + 3 * f), B4 = __ldg(p.rc_tri + 3 * f + 1), C4 = __ldg(p.rc_tri + 3 * f + 2);
            const F3 A = mk3(A4.x, A4.y, A4.z), B = mk3(B4.x, B4.y, B4.z), C3 = mk3(C4.x, C4.y, C4.z);
            const F3 dcp = sub3(qo, closest_pt_tri(qo, A, B, C3));
            const float d2 = dot(dcp, dcp);
            float pen = d2 < R2 ? R - sqrtf(d2) : 0.f;
            const float th = ray_tri(qo, nd, A, B, C3);
            if (th >= 0.f && th < R) pen = fmaxf(pen, R - th);
            if (pen > best) { best = pen; wn = cross3(sub3(B, A), sub3(C3, A)); won = true; }
          }
        } else if (sp + 2 <= 48) {
          stack[sp++] = __float_as_int(n0.w);        // inner node: left child, and the right child stored negated
          stack[sp++] = -__float_as_int(n1.w);       // (count > 0 marks a leaf; child indices are >= 1)
        }
      }
      if (won) {  // face normal of the winner of THIS object, object frame -> link frame
        const double nl = sqrt((double)wn.x * wn.x + (double)wn.y * wn.y + (double)wn.z * wn.z);
        if (nl > 0.0) bn = mulRT(RL, mulR(RO, D3{wn.x / nl, wn.y / nl, wn.z / nl}));
      }
    }
  }
  if (p.depth_rc) __stcs(p.depth_rc + gt, best);
  if (p.nrm_rc) { __stcs(p.nrm_rc + gt * 3, (float)bn.x); __stcs(p.nrm_rc + gt * 3 + 1, (float)bn.y); __stcs(p.nrm_rc + gt * 3 + 2, (float)bn.z); }
}

}  // namespace

unsigned long long ts_bank_elems_per_grid(int N) { return (unsigned long long)(N - 1) * (N - 1) * N; }

unsigned long long ts_step_smem_bytes(const TsStepParams& p) {
  return (unsigned long long)p.frames_per_group * p.K * sizeof(FrameS) + sizeof(float) * 2 * TS_BLOCK +
         (unsigned long long)p.s_bytes + sizeof(int) * TS_MAX_GROUP_PATCHES;
}

namespace {
template <bool SINGLE, int HM, bool FAST = false>
cudaError_t prep_one(int smem) {
  cudaError_t e = cudaFuncSetAttribute(ts_step_kernel<SINGLE, HM, FAST>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  // Ask for no more shared memory than TS_MIN_BLOCKS resident blocks need (+1 KB reserved per block): the
  // rest of the 228 KB stays L1, which serves the SDF gathers (measured: 1.51 -> 1.48 ms on config 5).
  const int carve = (int)((TS_MIN_BLOCKS * (smem + 1024LL) * 100 + 228 * 1024 - 1) / (228 * 1024)) + 2;
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(ts_step_kernel<SINGLE, HM, FAST>, cudaFuncAttributePreferredSharedMemoryCarveout, carve > 100 ? 100 : carve);
  return e;
}
template <bool SINGLE>
void launch_one(const TsStepParams& p, int hm, dim3 grid, size_t smem, cudaStream_t st) {
  switch (hm) {
    case TS_HYST_OFF: ts_step_kernel<SINGLE, TS_HYST_OFF><<<grid, TS_BLOCK, smem, st>>>(p); break;
    case TS_HYST_MAXWELL: ts_step_kernel<SINGLE, TS_HYST_MAXWELL><<<grid, TS_BLOCK, smem, st>>>(p); break;
    case TS_HYST_ASYM: ts_step_kernel<SINGLE, TS_HYST_ASYM><<<grid, TS_BLOCK, smem, st>>>(p); break;
    case 4 | TS_HYST_OFF: ts_step_kernel<SINGLE, 4 | TS_HYST_OFF><<<grid, TS_BLOCK, smem, st>>>(p); break;
    case 4 | TS_HYST_MAXWELL: ts_step_kernel<SINGLE, 4 | TS_HYST_MAXWELL><<<grid, TS_BLOCK, smem, st>>>(p); break;
    case 4 | TS_HYST_ASYM: ts_step_kernel<SINGLE, 4 | TS_HYST_ASYM><<<grid, TS_BLOCK, smem, st>>>(p); break;
    default: ts_step_kernel<SINGLE, -1><<<grid, TS_BLOCK, smem, st>>>(p); break;
  }
}
}  // namespace

// cudaFuncAttributeMaxDynamicSharedMemorySize and the carveout are per DEVICE, not per ctx: contexts with different
// shared-memory needs (K = 1 next to K = 8, say) share them, so the attribute is only ever RAISED to the running
// maximum of what any ctx on the device asked for (a later, smaller ctx must not shrink it under an earlier one).
int ts_prepare_kernels(int device, int smem_bytes) {
  static std::mutex mu;
  static int max_smem[64] = {0};
  std::lock_guard<std::mutex> lock(mu);
  const int d = device >= 0 && device < 64 ? device : 0;
  if (smem_bytes <= max_smem[d]) return 0;
  const int max_smem_bytes = smem_bytes;
  cudaError_t e = prep_one<true, -1>(max_smem_bytes);
  if (e == cudaSuccess) e = prep_one<true, -1, true>(max_smem_bytes);
  if (e == cudaSuccess) e = prep_one<true, TS_HYST_MAXWELL, true>(max_smem_bytes);
  if (e == cudaSuccess) e = prep_one<true, TS_HYST_ASYM, true>(max_smem_bytes);
  if (e == cudaSuccess) e = prep_one<true, 4 | TS_HYST_MAXWELL, true>(max_smem_bytes);
  if (e == cudaSuccess) e = prep_one<true, 4 | TS_HYST_ASYM, true>(max_smem_bytes);
  if (e == cudaSuccess) e = prep_one<true, TS_HYST_OFF>(max_smem_bytes);
  if (e == cudaSuccess) e = prep_one<true, TS_HYST_MAXWELL>(max_smem_bytes);
  if (e == cudaSuccess) e = prep_one<true, TS_HYST_ASYM>(max_smem_bytes);
  if (e == cudaSuccess) e = prep_one<true, 4 | TS_HYST_OFF>(max_smem_bytes);
  if (e == cudaSuccess) e = prep_one<true, 4 | TS_HYST_MAXWELL>(max_smem_bytes);
  if (e == cudaSuccess) e = prep_one<true, 4 | TS_HYST_ASYM>(max_smem_bytes);
  if (e == cudaSuccess) e = prep_one<false, 4 | TS_HYST_OFF>(max_smem_bytes);
  if (e == cudaSuccess) e = prep_one<false, 4 | TS_HYST_MAXWELL>(max_smem_bytes);
  if (e == cudaSuccess) e = prep_one<false, 4 | TS_HYST_ASYM>(max_smem_bytes);
  if (e == cudaSuccess) e = prep_one<false, -1>(max_smem_bytes);
  if (e == cudaSuccess) e = prep_one<false, TS_HYST_OFF>(max_smem_bytes);
  if (e == cudaSuccess) e = prep_one<false, TS_HYST_MAXWELL>(max_smem_bytes);
  if (e == cudaSuccess) e = prep_one<false, TS_HYST_ASYM>(max_smem_bytes);
  if (e == cudaSuccess) max_smem[d] = max_smem_bytes;
  return (int)e;
}

// fused_noise != 0: one launch does everything; otherwise the geometry kernel, and (noise on) ts_launch_noise.
// Launch with the programmatic-stream-serialization attribute: the grid may begin once every block of the kernel in
// front of it in the stream (ts_frames_kernel) has executed griddepcontrol.launch_dependents; its thread 0 waits for that
// grid's completion before it touches frames_g.  A predecessor that never triggers (an event record, a memcpy, another
// library's kernel) degrades this to a normal launch.
template <typename KernelT>
static int launch_dependent(KernelT kernel, dim3 grid, size_t smem, cudaStream_t stream, const TsStepParams& p) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = dim3(TS_BLOCK);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = TS_PDL ? 1 : 0;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  return (int)cudaLaunchKernelEx(&cfg, kernel, p);
}

int ts_launch_step(const TsStepParams& p, int fused_noise, void* stream) {
  if (p.E <= 0 || p.G <= 0 || p.G > 65535) return (int)cudaErrorInvalidConfiguration;
  const size_t smem = (size_t)ts_step_smem_bytes(p);
#if TS_GRID_GFAST
  const dim3 grid((unsigned)p.G, (unsigned)(p.E < 65535 ? p.E : 65535), (unsigned)((p.E + 65534) / 65535));
#else
  const dim3 grid((unsigned)p.E, (unsigned)p.G);
#endif
  const int hm = (p.noise_enable && fused_noise) ? (p.hyst_mode | (p.ext ? 4 : 0)) : -1;
  // the common full configuration has its own compile-time-specialised variants (see ts_step_kernel)
  const bool clean5 = p.K == 1 && p.inl && p.env_perm && p.mk_mma && p.contact && p.depth && p.ft && p.marker && p.prox;
  const bool fast = clean5 && p.ft_noisy && p.dead && ((hm & 3) == TS_HYST_ASYM || (hm & 3) == TS_HYST_MAXWELL);
  if (clean5 && hm == -1 && !p.noise_enable && !p.dead && !p.depth_pert)
    return launch_dependent(ts_step_kernel<true, -1, true>, grid, smem, (cudaStream_t)stream, p);
  else if (fast && hm == TS_HYST_ASYM) return launch_dependent(ts_step_kernel<true, TS_HYST_ASYM, true>, grid, smem, (cudaStream_t)stream, p);
  else if (fast && hm == TS_HYST_MAXWELL) return launch_dependent(ts_step_kernel<true, TS_HYST_MAXWELL, true>, grid, smem, (cudaStream_t)stream, p);
  else if (fast && hm == (4 | TS_HYST_ASYM)) return launch_dependent(ts_step_kernel<true, 4 | TS_HYST_ASYM, true>, grid, smem, (cudaStream_t)stream, p);
  else if (fast) return launch_dependent(ts_step_kernel<true, 4 | TS_HYST_MAXWELL, true>, grid, smem, (cudaStream_t)stream, p);
  else if (p.K == 1) launch_one<true>(p, hm, grid, smem, (cudaStream_t)stream);
  else launch_one<false>(p, hm, grid, smem, (cudaStream_t)stream);
  return (int)cudaGetLastError();
}

unsigned long long ts_frame_bytes() { return sizeof(FrameS); }

int ts_launch_frames(const TsStepParams& p, void* stream) {
  const long long n = (long long)p.E * p.P * p.K;
#if TS_PDL >= 2
  // Chained across steps: when the kernel in front of this one in the stream is the previous ts_step_kernel, this grid's
  // blocks may become resident once every block of it has fetched its frames; they wait at their top for it to complete
  // (griddepcontrol.wait), so only launch latency and ramp-up overlap.  Anything else in front (the caller's own kernels
  // writing the next poses, an event record, a copy) makes this an ordinary launch.
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)((n + 127) / 128));
  cfg.blockDim = dim3(128);
  cfg.dynamicSmemBytes = 0;
  cfg.stream = (cudaStream_t)stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  return (int)cudaLaunchKernelEx(&cfg, ts_frames_kernel, p);
#else
  ts_frames_kernel<<<(unsigned)((n + 127) / 128), 128, 0, (cudaStream_t)stream>>>(p);
  return (int)cudaGetLastError();
#endif
}

int ts_launch_shear(const TsStepParams& p, void* stream) {
  ts_shear_kernel<<<(unsigned)(p.E * p.P), 256, 0, (cudaStream_t)stream>>>(p);
  return (int)cudaGetLastError();
}

int ts_launch_reset_shear(const TsStepParams& p, const uint8_t* mask, void* stream) {
  const size_t n = (size_t)p.E * p.P * p.K * p.pc_np;
  ts_reset_shear_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(p, mask);
  return (int)cudaGetLastError();
}

int ts_launch_raycast(const TsStepParams& p, void* stream) {
  const long long n = (long long)p.E * p.T;
  ts_raycast_kernel<<<(unsigned)((n + 127) / 128), 128, 0, (cudaStream_t)stream>>>(p);
  return (int)cudaGetLastError();
}

int ts_launch_proxpc(const TsStepParams& p, void* stream) {
  const long long n = (long long)p.E * p.T;
  ts_proxpc_kernel<<<(unsigned)((n + 127) / 128), 128, 0, (cudaStream_t)stream>>>(p);
  return (int)cudaGetLastError();
}

int ts_launch_scalar_noise(const TsStepParams& p, void* stream) {
  const long long n = (long long)p.E * p.T + (long long)p.E * p.M;
  const unsigned blocks = (unsigned)((n + 255) / 256);
  cudaStream_t st = (cudaStream_t)stream;
  switch (p.hyst_mode) {
    case TS_HYST_MAXWELL: ts_scalar_noise_kernel<TS_HYST_MAXWELL><<<blocks, 256, 0, st>>>(p); break;
    case TS_HYST_ASYM: ts_scalar_noise_kernel<TS_HYST_ASYM><<<blocks, 256, 0, st>>>(p); break;
    default: ts_scalar_noise_kernel<TS_HYST_OFF><<<blocks, 256, 0, st>>>(p); break;
  }
  return (int)cudaGetLastError();
}

int ts_launch_reset_scalar(const TsStepParams& p, const uint8_t* mask, void* stream) {
  const long long n = (long long)p.E * (p.T > p.M ? p.T : p.M);
  ts_reset_scalar_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(p, mask);
  return (int)cudaGetLastError();
}

int ts_launch_noise(const TsStepParams& p, void* stream) {
  const dim3 grid((unsigned)p.E, (unsigned)p.G);
  cudaStream_t st = (cudaStream_t)stream;
  switch (p.hyst_mode | (p.ext ? 4 : 0)) {
    case TS_HYST_MAXWELL: ts_noise_kernel<TS_HYST_MAXWELL><<<grid, TS_BLOCK, 0, st>>>(p); break;
    case TS_HYST_ASYM: ts_noise_kernel<TS_HYST_ASYM><<<grid, TS_BLOCK, 0, st>>>(p); break;
    case 4 | TS_HYST_OFF: ts_noise_kernel<4 | TS_HYST_OFF><<<grid, TS_BLOCK, 0, st>>>(p); break;
    case 4 | TS_HYST_MAXWELL: ts_noise_kernel<4 | TS_HYST_MAXWELL><<<grid, TS_BLOCK, 0, st>>>(p); break;
    case 4 | TS_HYST_ASYM: ts_noise_kernel<4 | TS_HYST_ASYM><<<grid, TS_BLOCK, 0, st>>>(p); break;
    default: ts_noise_kernel<TS_HYST_OFF><<<grid, TS_BLOCK, 0, st>>>(p); break;
  }
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
  const long long threads = (long long)p.E * p.Tp;
  const long long blocks = (threads + 255) / 256;
  ts_reset_state_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(p, mask, thr, nh);
  return (int)cudaGetLastError();
}

// =======================================================================================
// ts_depth_static (include/ts.h): the contact-depth readout S1-S4 for analytic primitives with NO device allocation.
// It is the ctx-free variant of the frames-kernel -> step-kernel pair: the relative poses (the scratch that the ctx
// path keeps in the cudaMalloc'd frames_g) live in the file-scope array below, which every GPU that loads this library
// holds until the process exits.  Callers that cannot call cudaMalloc (graph capture, serving loops) use it.
// All calls on a device share the array; a call's pose kernel overwrites every record its depth kernel reads, so nothing
// in it needs to start at zero and nothing is cleared; two calls that overlap on the GPU (different streams) race on it.
// =======================================================================================
struct TsStaticFrame {   // 96 bytes: x_o = c + M x_j (link frame -> object frame), as FrameS::M / FrameS::c
  double M[9];
  double c[3];
};
static_assert(sizeof(TsStaticFrame) == 96 && TS_STATIC_SCRATCH_BYTES / sizeof(TsStaticFrame) == TS_STATIC_MAX_FRAMES,
              "static scratch layout");

// In host code this name is only a handle for cudaGetSymbolAddress; it is NOT a device address.
static __device__ __align__(256) unsigned char ts_static_scratch[TS_STATIC_SCRATCH_BYTES];

namespace {
// One thread per (env, link): M = R_O^T R_L, c = R_O^T (p_L - p_O) in double (Eq. 1; p_L - p_O formed before
// rotating, as in build_frame_row).
__global__ void __launch_bounds__(128) ts_static_frames_kernel(TsStaticFrame* __restrict__ fr, int E, int L, const float* __restrict__ link_pos,
                                                               const float* __restrict__ link_quat, const float* __restrict__ obj_pos,
                                                               const float* __restrict__ obj_quat) {
  const int gt = blockIdx.x * blockDim.x + threadIdx.x;
  if (gt >= E * L) return;
  const int e = gt / L;
  double RL[9], RO[9];
  quat_Rd(link_quat + (size_t)gt * 4, RL);
  quat_Rd(obj_quat + (size_t)e * 4, RO);
  const D3 d = ld3d(link_pos + (size_t)gt * 3) - ld3d(obj_pos + (size_t)e * 3);
  TsStaticFrame F;
#pragma unroll
  for (int r = 0; r < 3; ++r) {   // row r of R_O^T = column r of R_O
    const double o0 = RO[r], o1 = RO[3 + r], o2 = RO[6 + r];
#pragma unroll
    for (int c = 0; c < 3; ++c) F.M[r * 3 + c] = fma(o0, RL[c], fma(o1, RL[3 + c], o2 * RL[6 + c]));
    F.c[r] = fma(o0, d.x, fma(o1, d.y, o2 * d.z));
  }
  fr[gt] = F;
}

// The primitive cases of phi_d (O2), same expressions.
__device__ __forceinline__ double phi_prim_d(int type, float4 prm, D3 x) {
  if (type == TS_GEOM_SPHERE) return dsqrt_n(dot(x, x)) - (double)prm.x;
  if (type == TS_GEOM_BOX) {
    const double wx = fabs(x.x) - (double)prm.x, wy = fabs(x.y) - (double)prm.y, wz = fabs(x.z) - (double)prm.z;
    const double px = fmax(wx, 0.0), py = fmax(wy, 0.0), pz = fmax(wz, 0.0);
    return dsqrt_n(fma(px, px, fma(py, py, pz * pz))) + fmin(fmax(wx, fmax(wy, wz)), 0.0);
  }
  if (type == TS_GEOM_CAPSULE) {
    const double h = (double)prm.y;
    const double zc = fmin(fmax(x.z, -h), h);
    const D3 y = D3{x.x, x.y, x.z - zc};
    return dsqrt_n(dot(y, y)) - (double)prm.x;
  }
  return __longlong_as_double(0x7ff0000000000000LL);   // no object (or a type this entry point does not serve): depth 0
}

// One thread per (env, taxel): d = [R_j - phi(c + M x_j)]_+ (Eq. 2), rounded once.
__global__ void __launch_bounds__(256) ts_static_depth_kernel(const TsStaticFrame* __restrict__ fr, int E, int L, int T,
                                                              const float* __restrict__ taxel_pos, const float* __restrict__ taxel_radius,
                                                              const int32_t* __restrict__ taxel_link, const int32_t* __restrict__ geom_type,
                                                              const float* __restrict__ geom_params, float* __restrict__ depth) {
  const long long gt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gt >= (long long)E * T) return;
  const int e = (int)(gt / T), j = (int)(gt - (long long)e * T);
  const float Rj = __ldg(taxel_radius + j);
  const int link = __ldg(taxel_link + j);
  float d = 0.f;
  if (Rj > 0.f && link >= 0 && link < L) {
    const TsStaticFrame& F = fr[(size_t)e * L + link];
    const D3 xj = ld3d(taxel_pos + (size_t)j * 3);
    const D3 x = ldv(F.c) + mulR(F.M, xj);
    const float4 prm = __ldg(reinterpret_cast<const float4*>(geom_params) + e);
    const double dd = (double)Rj - phi_prim_d(__ldg(geom_type + e), prm, x);
    d = dd > 0.0 ? (float)dd : 0.f;
  }
  depth[gt] = d;
}

// Device address of ts_static_scratch, looked up once per device with that device current.
std::mutex g_static_mu;
void* g_static_ptr[64] = {};
}  // namespace

int ts_static_depth_launch(int E, int L, int T, const float* taxel_pos, const float* taxel_radius, const int32_t* taxel_link,
                           const float* link_pos, const float* link_quat, const float* obj_pos, const float* obj_quat,
                           const int32_t* geom_type, const float* geom_params, float* depth, void* stream) {
  if ((long long)E * L > (long long)TS_STATIC_MAX_FRAMES) return (int)cudaErrorInvalidValue;   // the caller checked already
  int dev = -1;
  cudaError_t err = cudaGetDevice(&dev);
  if (err != cudaSuccess) return (int)err;
  if (dev < 0 || dev >= 64) return (int)cudaErrorInvalidDevice;
  void* ptr = nullptr;
  {
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_ptr[dev]) {   // set-up, once per device: the symbol's address ON THIS DEVICE (no allocation happens here)
      void* q = nullptr;
      err = cudaGetSymbolAddress(&q, ts_static_scratch);
      if (err != cudaSuccess) return (int)err;
      g_static_ptr[dev] = q;
    }
    ptr = g_static_ptr[dev];
  }
  TsStaticFrame* fr = static_cast<TsStaticFrame*>(ptr);
  const cudaStream_t st = (cudaStream_t)stream;
  ts_static_frames_kernel<<<(unsigned)((E * L + 127) / 128), 128, 0, st>>>(fr, E, L, link_pos, link_quat, obj_pos, obj_quat);
  err = cudaGetLastError();
  if (err != cudaSuccess) return (int)err;
  const long long n = (long long)E * T;
  ts_static_depth_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(fr, E, L, T, taxel_pos, taxel_radius, taxel_link, geom_type,
                                                                      geom_params, depth);
  return (int)cudaGetLastError();
}
