// A/B experiment (not on the product path): SDF queries served from a per-patch BRICK staged in shared memory by TMA
// (cp.async.bulk.tensor.3d, SASS UTMALDG) against the product's gather path (quad-layout bank, two LDG.128 per
// evaluation).  BASELINE north_star names "SDF grids staged by TMA or shared memory"; this measures that design on the
// shapes of configs 3 and 5.  Both kernels run the same work: for every taxel of every query patch the first SDF query
// and a bounded march of `steps` evaluations along the patch normal, all in the object frame, fp32, interior points.
//
//   gather: thread per taxel; cell index -> Q[(j (N-1) + i) N + k], two float4 loads per evaluation (L1 / L2 hits).
//   brick : block per patch; thread 0 bounds the patch's march volume by an axis-aligned box of BXYZ^3 voxels and issues
//           ONE 3-D tensor copy of it from the linear bank; after the mbarrier flips, every evaluation reads its 8
//           corners from shared memory; an evaluation that leaves the brick falls back to the gather.
//
// C ABI: brick_ab_run(...) returns 0 on success; times are CUDA-event means over `reps` launches.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <vector>

namespace {

struct Patch {
  float c[3];      // pad centre, object frame [m]
  float u[3], v[3], n[3];
  int grid;
};

__device__ __forceinline__ float trilerp8(const float c[8], float fx, float fy, float fz) {
  const float a0 = fmaf(fx, c[1] - c[0], c[0]), a1 = fmaf(fx, c[3] - c[2], c[2]);
  const float b0 = fmaf(fx, c[5] - c[4], c[4]), b1 = fmaf(fx, c[7] - c[6], c[6]);
  const float lo = fmaf(fy, a1 - a0, a0), hi = fmaf(fy, b1 - b0, b0);
  return fmaf(fz, hi - lo, lo);
}

__device__ __forceinline__ float gather_eval(const float4* quad, int N, size_t gstride, int g, float ux, float uy, float uz) {
  const int i = (int)ux, j = (int)uy, k = (int)uz;
  const float4* q = quad + (size_t)g * gstride + ((size_t)(j * (N - 1) + i) * N + k);
  const float4 A = __ldg(q), B = __ldg(q + 1);
  const float c[8] = {A.x, A.y, A.z, A.w, B.x, B.y, B.z, B.w};
  return trilerp8(c, ux - (float)i, uy - (float)j, uz - (float)k);
}

__device__ __forceinline__ void taxel_start(const Patch& p, int nu, int nv, float pitch, int t, float inv_voxel, float half, float* u0, float* du) {
  const int iu = t % nu, iv = t / nu;
  const float su = ((float)iu + 0.5f - 0.5f * (float)nu) * pitch, sv = ((float)iv + 0.5f - 0.5f * (float)nv) * pitch;
  for (int a = 0; a < 3; ++a) {
    u0[a] = fmaf(p.c[a] + su * p.u[a] + sv * p.v[a], inv_voxel, half);
    du[a] = p.n[a] * inv_voxel;
  }
}

__global__ void gather_kernel(const Patch* patches, int Q, int nu, int nv, float pitch, const float4* quad, int N, size_t gstride,
                              float voxel, float r_prox, int steps, float* out) {
  const int gt = blockIdx.x * blockDim.x + threadIdx.x;
  const int per = nu * nv;
  if (gt >= Q * per) return;
  const Patch p = patches[gt / per];
  float u0[3], du[3];
  taxel_start(p, nu, nv, pitch, gt % per, 1.f / voxel, 0.5f * (float)(N - 1), u0, du);
  float t = 0.f;
  for (int it = 0; it < steps; ++it) {
    const float s = gather_eval(quad, N, gstride, p.grid, fmaf(t, du[0], u0[0]), fmaf(t, du[1], u0[1]), fmaf(t, du[2], u0[2]));
    t = fminf(t + fmaxf(s, 0.f), r_prox);
  }
  out[gt] = r_prox - t;
}

[[maybe_unused]] __device__ __forceinline__ uint32_t s32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

template <int B>
__global__ void brick_kernel(const CUtensorMap* __restrict__ tmap_g, const float* lin, const Patch* patches, int Q, int nu, int nv, float pitch,
                             const float4* quad, int N, size_t gstride, float voxel, float r_prox, int steps, float* out,
                             unsigned* fallbacks) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float* brick = reinterpret_cast<float*>((reinterpret_cast<uintptr_t>(smem_raw) + 127) & ~(uintptr_t)127);   // [B][B][B], x fastest; TMA wants 128-byte alignment
  __shared__ __align__(8) uint64_t bar;   // unused in the -DBRICK_NO_TMA arm
  (void)bar;
  __shared__ int org[3];
  const int q = blockIdx.x, tid = threadIdx.x, per = nu * nv;
  const Patch p = patches[q];
  const float inv_voxel = 1.f / voxel, half = 0.5f * (float)(N - 1);
  if (tid == 0) {
    // bounding box (voxel coordinates) of the pad corners and of the pad corners moved by r_prox along the normal
    float lo[3] = {1e30f, 1e30f, 1e30f};
    const float hu = 0.5f * (float)nu * pitch, hv = 0.5f * (float)nv * pitch;
    for (int s = 0; s < 8; ++s)
      for (int a = 0; a < 3; ++a) {
        const float x = p.c[a] + ((s & 1) ? hu : -hu) * p.u[a] + ((s & 2) ? hv : -hv) * p.v[a] + ((s & 4) ? r_prox : 0.f) * p.n[a];
        lo[a] = fminf(lo[a], fmaf(x, inv_voxel, half));
      }
    for (int a = 0; a < 3; ++a) org[a] = min(max((int)floorf(lo[a]), 0), N - B);   // N and B are multiples of 4
    org[0] &= ~3;   // 16-byte aligned row starts for the bulk copies (the box was sized with that slack)
#ifndef BRICK_NO_TMA
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(s32(&bar)) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(s32(&bar)), "r"((unsigned)(B * B * B * 4)) : "memory");
#endif
  }
  __syncthreads();
#ifdef BRICK_NO_TMA
  // third arm: the same brick filled by plain cooperative loads from the linear bank (no TMA)
  for (int idx = tid; idx < B * B * B; idx += blockDim.x) {
    const int i = idx % B, j = (idx / B) % B, k = idx / (B * B);
    brick[idx] = __ldg(lin + (size_t)p.grid * N * N * N + ((size_t)(org[2] + k) * N + (org[1] + j)) * N + (org[0] + i));
  }
  __syncthreads();
#else
  // TMA arm: B * B bulk copies of one brick row (B floats) each, cp.async.bulk (SASS UBLKCP), all completing on one
  // mbarrier.  (The single-instruction form, cp.async.bulk.tensor.4d on a cuTensorMapEncodeTiled descriptor -- SASS
  // UTMALDG.4D -- was built first and faulted with "illegal instruction" on this pool's driver whether the descriptor sat
  // in the parameter space or in global memory; see profiles/r02_brick_ab.md.  TMAP arm kept under BRICK_TENSOR_MAP.)
#ifdef BRICK_TENSOR_MAP
  if (tid == 0)
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 ::"r"(s32(brick)), "l"(reinterpret_cast<uint64_t>(tmap_g)), "r"(org[0]), "r"(org[1]), "r"(org[2]), "r"(p.grid), "r"(s32(&bar)) : "memory");
#else
  for (int row = tid; row < B * B; row += blockDim.x) {
    const int j = row % B, k = row / B;
    const float* src = lin + (size_t)p.grid * N * N * N + ((size_t)(org[2] + k) * N + (org[1] + j)) * N + org[0];
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(s32(brick + row * B)), "l"(src), "r"((unsigned)(B * 4)), "r"(s32(&bar)) : "memory");
  }
#endif
  asm volatile(
      "{\n.reg .pred p;\nW_%=:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], 0;\n@!p bra W_%=;\n}\n" ::"r"(s32(&bar)) : "memory");
#endif
  if (tid >= per) return;
  float u0[3], du[3];
  taxel_start(p, nu, nv, pitch, tid, inv_voxel, half, u0, du);
  const int ox = org[0], oy = org[1], oz = org[2];
  float t = 0.f;
  unsigned fb = 0;
  for (int it = 0; it < steps; ++it) {
    const float ux = fmaf(t, du[0], u0[0]), uy = fmaf(t, du[1], u0[1]), uz = fmaf(t, du[2], u0[2]);
    const int i = (int)ux - ox, j = (int)uy - oy, k = (int)uz - oz;
    float s;
    if ((unsigned)i < (unsigned)(B - 1) && (unsigned)j < (unsigned)(B - 1) && (unsigned)k < (unsigned)(B - 1)) {
      const float* b0 = brick + (k * B + j) * B + i;
      const float c[8] = {b0[0], b0[1], b0[B], b0[B + 1], b0[B * B], b0[B * B + 1], b0[B * B + B], b0[B * B + B + 1]};
      // quad order of the product: (c000, c100, c010, c110), (c001, c101, c011, c111) with k the fast index of the bank
      const float cq[8] = {c[0], c[1], c[2], c[3], c[4], c[5], c[6], c[7]};
      s = trilerp8(cq, ux - (float)(i + ox), uy - (float)(j + oy), uz - (float)(k + oz));
    } else {
      s = gather_eval(quad, N, gstride, p.grid, ux, uy, uz);
      ++fb;
    }
    t = fminf(t + fmaxf(s, 0.f), r_prox);
  }
  out[q * per + tid] = r_prox - t;
  if (fb) atomicAdd(fallbacks, fb);
}

__global__ void retile(const float* src, float4* dst, int G, int N) {
  const size_t per = (size_t)(N - 1) * (N - 1) * N, total = per * G;
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

}  // namespace

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

#define CK(x)                                                                     \
  do {                                                                            \
    cudaError_t e_ = (x);                                                         \
    if (e_ != cudaSuccess) { std::fprintf(stderr, "line %d: %s: %s\n", __LINE__, #x, cudaGetErrorString(e_)); return 1; } \
  } while (0)

template <int B>
static int run_brick(const CUtensorMap* tmap, const float* d_lin, const Patch* d_p, int Q, int nu, int nv, float pitch, const float4* d_quad, int N,
                     size_t gstride, float voxel, float r_prox, int steps, float* d_out, unsigned* d_fb, int reps, float* ms) {
  const size_t smem = sizeof(float) * B * B * B + 128;
  CK(cudaFuncSetAttribute(brick_kernel<B>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  cudaEvent_t e0, e1;
  CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
  const int threads = ((nu * nv + 31) / 32) * 32;
  for (int w = 0; w < 3; ++w) brick_kernel<B><<<Q, threads, smem>>>(tmap, d_lin, d_p, Q, nu, nv, pitch, d_quad, N, gstride, voxel, r_prox, steps, d_out, d_fb);
  CK(cudaMemset(d_fb, 0, 4));
  CK(cudaEventRecord(e0));
  for (int r = 0; r < reps; ++r) brick_kernel<B><<<Q, threads, smem>>>(tmap, d_lin, d_p, Q, nu, nv, pitch, d_quad, N, gstride, voxel, r_prox, steps, d_out, d_fb);
  CK(cudaEventRecord(e1));
  CK(cudaEventSynchronize(e1));
  CK(cudaGetLastError());
  CK(cudaEventElapsedTime(ms, e0, e1));
  *ms /= (float)reps;
  return 0;
}

extern "C" int brick_ab_run(const float* bank_host, int G, int N, float voxel, const float* patches_host /* [Q,13]: c, u, v, n, grid */,
                            int Q, int nu, int nv, float pitch, float r_prox, int steps, int brick, int reps, float* out_gather,
                            float* out_brick, float* ms /* [2] */, unsigned* fallbacks) {
  std::vector<Patch> hp(Q);
  for (int q = 0; q < Q; ++q) {
    const float* s = patches_host + 13 * q;
    for (int a = 0; a < 3; ++a) { hp[q].c[a] = s[a]; hp[q].u[a] = s[3 + a]; hp[q].v[a] = s[6 + a]; hp[q].n[a] = s[9 + a]; }
    hp[q].grid = (int)s[12];
  }
  float *d_lin = nullptr, *d_og = nullptr, *d_ob = nullptr;
  float4* d_quad = nullptr;
  Patch* d_p = nullptr;
  unsigned* d_fb = nullptr;
  const size_t lin = (size_t)G * N * N * N, gstride = (size_t)(N - 1) * (N - 1) * N, nt = (size_t)Q * nu * nv;
  CK(cudaMalloc(&d_lin, lin * 4)); CK(cudaMalloc(&d_quad, gstride * G * 16)); CK(cudaMalloc(&d_p, sizeof(Patch) * Q));
  CK(cudaMalloc(&d_og, nt * 4)); CK(cudaMalloc(&d_ob, nt * 4)); CK(cudaMalloc(&d_fb, 4));
  CK(cudaMemcpy(d_lin, bank_host, lin * 4, cudaMemcpyHostToDevice));
  CK(cudaMemcpy(d_p, hp.data(), sizeof(Patch) * Q, cudaMemcpyHostToDevice));
  retile<<<148 * 8, 256>>>(d_lin, d_quad, G, N);
  CK(cudaDeviceSynchronize());
  // gather path
  cudaEvent_t e0, e1;
  CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
  const int blocks = (int)((nt + 255) / 256);
  for (int w = 0; w < 3; ++w) gather_kernel<<<blocks, 256>>>(d_p, Q, nu, nv, pitch, d_quad, N, gstride, voxel, r_prox, steps, d_og);
  CK(cudaEventRecord(e0));
  for (int r = 0; r < reps; ++r) gather_kernel<<<blocks, 256>>>(d_p, Q, nu, nv, pitch, d_quad, N, gstride, voxel, r_prox, steps, d_og);
  CK(cudaEventRecord(e1));
  CK(cudaEventSynchronize(e1));
  CK(cudaGetLastError());
  CK(cudaEventElapsedTime(&ms[0], e0, e1));
  ms[0] /= (float)reps;
  // brick path: 4-D tensor map (x, y, z, grid) over the LINEAR bank, box brick^3 x 1
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  CK(cudaGetDriverEntryPointByVersion("cuTensorMapEncodeTiled", &fn, 12000, cudaEnableDefault, &qres));
  if (!fn || qres != cudaDriverEntryPointSuccess) { std::fprintf(stderr, "cuTensorMapEncodeTiled not available\n"); return 2; }
  CUtensorMap tmap;
  const cuuint64_t dims[4] = {(cuuint64_t)N, (cuuint64_t)N, (cuuint64_t)N, (cuuint64_t)G};
  const cuuint64_t strides[3] = {(cuuint64_t)N * 4, (cuuint64_t)N * N * 4, (cuuint64_t)N * N * N * 4};
  const cuuint32_t box[4] = {(cuuint32_t)brick, (cuuint32_t)brick, (cuuint32_t)brick, 1};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  const CUresult cr = ((EncodeTiledFn)fn)(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, d_lin, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                          CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (cr != CUDA_SUCCESS) { std::fprintf(stderr, "cuTensorMapEncodeTiled failed: %d\n", (int)cr); return 3; }
  int rc = 0;
  CUtensorMap* d_tmap = nullptr;   // the descriptor lives in global memory (64-byte aligned by cudaMalloc)
  CK(cudaMalloc(&d_tmap, sizeof(CUtensorMap)));
  CK(cudaMemcpy(d_tmap, &tmap, sizeof(CUtensorMap), cudaMemcpyHostToDevice));
  if (brick == 16) rc = run_brick<16>(d_tmap, d_lin, d_p, Q, nu, nv, pitch, d_quad, N, gstride, voxel, r_prox, steps, d_ob, d_fb, reps, &ms[1]);
  else if (brick == 24) rc = run_brick<24>(d_tmap, d_lin, d_p, Q, nu, nv, pitch, d_quad, N, gstride, voxel, r_prox, steps, d_ob, d_fb, reps, &ms[1]);
  else if (brick == 32) rc = run_brick<32>(d_tmap, d_lin, d_p, Q, nu, nv, pitch, d_quad, N, gstride, voxel, r_prox, steps, d_ob, d_fb, reps, &ms[1]);
  else rc = 4;
  if (rc) return rc;
  CK(cudaMemcpy(out_gather, d_og, nt * 4, cudaMemcpyDeviceToHost));
  CK(cudaMemcpy(out_brick, d_ob, nt * 4, cudaMemcpyDeviceToHost));
  CK(cudaMemcpy(fallbacks, d_fb, 4, cudaMemcpyDeviceToHost));
  cudaFree(d_lin); cudaFree(d_quad); cudaFree(d_p); cudaFree(d_og); cudaFree(d_ob); cudaFree(d_fb);
  return 0;
}
