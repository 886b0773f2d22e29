// mt_probe_field.cu — the three ways north_star subsystem (5) names for serving the trilinear field corners ("texture/L2
// or TMA-staged tiles"; "the builder must measure all three"), measured side by side on ONE access
// pattern that is the step loop's own at its best for staging: the 256 lanes of a CTA sit in a 4 x 4 block of cell columns
// of a padded 202 x 202 x 66 grid of 32-byte x-pair records (one z-slab of config 3), walk 64 layers in
// lock-step and fetch, per layer, the four records of a trilinear corner set: (x, y, z), (x, y+1, z), (x, y, z+1),
// (x, y+1, z+1).
//   LDG   what the transport kernels do: four ld.global.nc.v8.f32 through L1/L2.
//   TEX   the same records point-sampled (no filtering: 9-bit weights would break parity) from a 3D float4 texture,
//         two fetches per record.
//   TMA   the CTA's 12 x 12-column window staged in shared memory nine layers at a time by cp.async.bulk.tensor
//         (two stages, mbarrier hand-over), corners read from shared memory.
// Behind mt_probe_field_paths() in include/muon_transport.h; numbers in DESIGN.md §7 / profiles/r2_summary.md.  Not on
// the transport path.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/muon_probes.h"
#include "../../include/muon_transport.h"      // (the MT_ERR_* codes)

namespace {

constexpr int PX = 202, PY = 202, PZ = 66;       // padded grid (records)
constexpr int BX = 12, BY = 12, BZ = 9;          // TMA box: window of columns x layers per stage (8 new layers + 1 shared)
constexpr int ZSTEPS = 64;
constexpr int STAGE_FLOATS = 8 * BX * BY * BZ;   // 41 472 B per stage

struct Rec { float v[8]; };

// where the CTA's window starts, and where a lane sits inside it (drifting one cell in x every 16 layers)
__device__ __forceinline__ void place(int cta, int tid, int& x0, int& y0, int& lx, int& ly) {
  const uint32_t h = (uint32_t)cta * 2654435761u;
  x0 = (int)(h % (uint32_t)(PX - BX));
  y0 = (int)((h >> 12) % (uint32_t)(PY - BY));
  const int lane = tid & 31, warp = tid >> 5;
  lx = (lane & 3) + (warp & 1) * 2;               // 0..5
  ly = ((lane >> 2) & 3) + ((warp >> 1) & 1) * 2 + ((lane >> 4) & 1) * 4;   // 0..9
}

__device__ __forceinline__ float use(const Rec& r) { return ((r.v[0] + r.v[1]) + (r.v[2] + r.v[3])) + ((r.v[4] + r.v[5]) + (r.v[6] + r.v[7])); }
__device__ __forceinline__ float use4(const float4& a) { return (a.x + a.y) + (a.z + a.w); }

__device__ __forceinline__ Rec ldg_rec(const Rec* p) {
  Rec r;
  asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=f"(r.v[0]), "=f"(r.v[1]), "=f"(r.v[2]), "=f"(r.v[3]), "=f"(r.v[4]), "=f"(r.v[5]), "=f"(r.v[6]), "=f"(r.v[7])
               : "l"(p));
  return r;
}

__global__ void __launch_bounds__(256) field_ldg_kernel(const Rec* __restrict__ grid, float* sink) {
  int x0, y0, lx, ly;
  place(blockIdx.x, threadIdx.x, x0, y0, lx, ly);
  float acc = 0.0f;
  for (int z = 0; z < ZSTEPS; ++z) {
    const int x = x0 + lx + (z >> 4), y = y0 + ly;
    const Rec* p = grid + ((size_t)z * PY + y) * PX + x;
    const Rec a = ldg_rec(p), b = ldg_rec(p + PX), c = ldg_rec(p + (size_t)PX * PY), d = ldg_rec(p + (size_t)PX * PY + PX);
    acc += use(a) + use(b) + use(c) + use(d);
  }
  if (acc == 0.12345f) sink[0] = acc;
}

__global__ void __launch_bounds__(256) field_tex_kernel(cudaTextureObject_t tex, float* sink) {
  int x0, y0, lx, ly;
  place(blockIdx.x, threadIdx.x, x0, y0, lx, ly);
  float acc = 0.0f;
  for (int z = 0; z < ZSTEPS; ++z) {
    const float x = (float)(2 * (x0 + lx + (z >> 4))), y = (float)(y0 + ly), zf = (float)z;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const float yy = y + (float)(c & 1), zz = zf + (float)(c >> 1);
      const float4 lo = tex3D<float4>(tex, x, yy, zz), hi = tex3D<float4>(tex, x + 1.0f, yy, zz);
      acc += use4(lo) + use4(hi);
    }
  }
  if (acc == 0.12345f) sink[0] = acc;
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__global__ void __launch_bounds__(256) field_tma_kernel(const __grid_constant__ CUtensorMap tmap, float* sink) {
  extern __shared__ __align__(128) float tile[];                 // [2][BZ][BY][BX][8]
  __shared__ __align__(8) uint64_t full[2];
  int x0, y0, lx, ly;
  place(blockIdx.x, threadIdx.x, x0, y0, lx, ly);
  const uint32_t bar0 = smem_u32(&full[0]), bar1 = smem_u32(&full[1]);
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar0));
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar1));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  auto issue = [&](int stage, int z_first) {
    const uint32_t bar = stage ? bar1 : bar0, dst = smem_u32(tile + (size_t)stage * STAGE_FLOATS);
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"((uint32_t)(STAGE_FLOATS * 4)) : "memory");
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 ::"r"(dst), "l"(&tmap), "r"(0), "r"(x0), "r"(y0), "r"(z_first), "r"(bar) : "memory");
  };
  if (threadIdx.x == 0) { issue(0, 0); issue(1, 8); }
  float acc = 0.0f;
  for (int chunk = 0; chunk < ZSTEPS / 8; ++chunk) {
    const int stage = chunk & 1;
    const uint32_t bar = stage ? bar1 : bar0, parity = (uint32_t)((chunk >> 1) & 1);
    asm volatile(
        "{\n.reg .pred p;\nWAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\nbra WAIT_%=;\nDONE_%=:\n}\n" ::"r"(bar), "r"(parity) : "memory");
    const float* t = tile + (size_t)stage * STAGE_FLOATS;
#pragma unroll 2
    for (int dz = 0; dz < 8; ++dz) {
      const int z = chunk * 8 + dz;
      const int x = lx + (z >> 4), y = ly;
      const float4* p = reinterpret_cast<const float4*>(t + (((size_t)dz * BY + y) * BX + x) * 8);
      const int sy = BX * 2, sz = BX * BY * 2;                   // strides in float4
      const float4 a0 = p[0], a1 = p[1], b0 = p[sy], b1 = p[sy + 1], c0 = p[sz], c1 = p[sz + 1], d0 = p[sz + sy], d1 = p[sz + sy + 1];
      acc += (use4(a0) + use4(a1)) + (use4(b0) + use4(b1)) + (use4(c0) + use4(c1)) + (use4(d0) + use4(d1));
    }
    __syncthreads();                                            // every warp is done with this stage
    if (threadIdx.x == 0 && chunk + 2 < ZSTEPS / 8) issue(stage, (chunk + 2) * 8);
  }
  if (acc == 0.12345f) sink[0] = acc;
}

template <class F> cudaError_t best_ms(F&& launch, float* out) {
  cudaEvent_t e0, e1;
  cudaError_t e = cudaEventCreate(&e0);
  if (e != cudaSuccess) return e;
  e = cudaEventCreate(&e1);
  if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
  *out = 1e30f;
  for (int r = 0; r < 4 && e == cudaSuccess; ++r) {
    cudaEventRecord(e0, 0);
    launch();
    cudaEventRecord(e1, 0);
    e = cudaEventSynchronize(e1);
    float ms = 0.0f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (e == cudaSuccess && r > 0 && ms < *out) *out = ms;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  if (e == cudaSuccess) e = cudaGetLastError();
  return e;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

}  // namespace

extern "C" int mt_probe_field_paths(int cuda_device, mt_field_paths* out) {
  if (!out) return MT_ERR_INVALID_ARG;
  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || cuda_device < 0 || cuda_device >= n_dev) { cudaGetLastError(); return MT_ERR_CUDA; }
  int prev = 0;
  cudaGetDevice(&prev);
  cudaSetDevice(cuda_device);
  int sms = 0;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, cuda_device);
  const int grid = sms * 3 * 16;                                  // 16 windows per resident CTA slot
  const double records = (double)grid * 256.0 * ZSTEPS * 4.0;
  const size_t n_rec = (size_t)PX * PY * PZ;
  Rec* d_grid = nullptr;
  float* sink = nullptr;
  cudaArray_t arr = nullptr;
  cudaTextureObject_t tex = 0;
  int rc = MT_OK;
  out->ldg_records_per_s = out->tex_records_per_s = out->tma_records_per_s = 0.0;
  out->records_per_launch = records;
  do {
    if (cudaMalloc(&d_grid, n_rec * sizeof(Rec)) != cudaSuccess || cudaMalloc(&sink, 256) != cudaSuccess) { rc = MT_ERR_NOMEM; break; }
    if (cudaMemset(d_grid, 0, n_rec * sizeof(Rec)) != cudaSuccess) { rc = MT_ERR_CUDA; break; }
    float ms = 0.0f;
    // ---- LDG
    if (best_ms([&] { field_ldg_kernel<<<grid, 256>>>(d_grid, sink); }, &ms) != cudaSuccess) { rc = MT_ERR_CUDA; break; }
    out->ldg_records_per_s = records / (ms * 1e-3);
    // ---- TEX: the same bytes as a 3D float4 array, two texels per record
    cudaChannelFormatDesc fd = cudaCreateChannelDesc<float4>();
    if (cudaMalloc3DArray(&arr, &fd, make_cudaExtent(2 * PX, PY, PZ)) != cudaSuccess) { rc = MT_ERR_NOMEM; break; }
    cudaMemcpy3DParms cp = {};
    cp.srcPtr = make_cudaPitchedPtr(d_grid, (size_t)2 * PX * sizeof(float4), 2 * PX, PY);
    cp.dstArray = arr;
    cp.extent = make_cudaExtent(2 * PX, PY, PZ);
    cp.kind = cudaMemcpyDeviceToDevice;
    if (cudaMemcpy3D(&cp) != cudaSuccess) { rc = MT_ERR_CUDA; break; }
    cudaResourceDesc rd = {};
    rd.resType = cudaResourceTypeArray;
    rd.res.array.array = arr;
    cudaTextureDesc td = {};
    td.addressMode[0] = td.addressMode[1] = td.addressMode[2] = cudaAddressModeClamp;
    td.filterMode = cudaFilterModePoint;
    td.readMode = cudaReadModeElementType;
    td.normalizedCoords = 0;
    if (cudaCreateTextureObject(&tex, &rd, &td, nullptr) != cudaSuccess) { rc = MT_ERR_CUDA; break; }
    if (best_ms([&] { field_tex_kernel<<<grid, 256>>>(tex, sink); }, &ms) != cudaSuccess) { rc = MT_ERR_CUDA; break; }
    out->tex_records_per_s = records / (ms * 1e-3);
    // ---- TMA: 4-D tensor map {8 floats, x, y, z}, box {8, BX, BY, BZ}
    EncodeTiledFn encode = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", (void**)&encode, cudaEnableDefault, &qres) != cudaSuccess || !encode) {
      cudaGetLastError();
      break;                                                     // tma_records_per_s stays 0: not available
    }
    CUtensorMap tmap;
    const cuuint64_t gdim[4] = {8, (cuuint64_t)PX, (cuuint64_t)PY, (cuuint64_t)PZ};
    const cuuint64_t gstride[3] = {32, (cuuint64_t)32 * PX, (cuuint64_t)32 * PX * PY};
    const cuuint32_t box[4] = {8, BX, BY, BZ}, estr[4] = {1, 1, 1, 1};
    if (encode(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, d_grid, gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) break;
    const size_t smem = (size_t)2 * STAGE_FLOATS * sizeof(float);
    if (cudaFuncSetAttribute((const void*)field_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) { rc = MT_ERR_CUDA; break; }
    if (best_ms([&] { field_tma_kernel<<<grid, 256, smem>>>(tmap, sink); }, &ms) != cudaSuccess) { rc = MT_ERR_CUDA; break; }
    out->tma_records_per_s = records / (ms * 1e-3);
  } while (0);
  if (tex) cudaDestroyTextureObject(tex);
  if (arr) cudaFreeArray(arr);
  if (d_grid) cudaFree(d_grid);
  if (sink) cudaFree(sink);
  cudaSetDevice(prev);
  return rc;
}
