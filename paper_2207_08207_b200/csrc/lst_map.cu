// lst_map.cu -- module-map builder [B] (DESIGN.md section 1 [B]): the step before the hot path.
//
// For every module A, every module B of the next layer is tested against the closed-form envelope of the
// pT >= pt_min helices that leave A's edges (B1-B4, binary64, no FMA contraction: this file is compiled with
// --fmad=false like the rest of the library).  One block per source module; its threads take the candidate
// modules in ascending order, 256 at a time, and an ordered block-level compaction (ballot + scan of the warp
// counts) writes the row ascending.  Two passes (count, then fill) around one exclusive scan of the row
// lengths on the host: the map is built once per geometry, its size (70 k entries) is known only afterwards.
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>
#include <vector>

#include "../../include/lst.h"

namespace {

struct MapGeom {
  int n;
  const signed char* layer;
  const double *phi, *rho, *gap, *hw, *zlo, *zhi;
};

__device__ __forceinline__ bool connected(const MapGeom& g, const lst_map_params& p, int A, int B) {
  if (g.layer[B] != g.layer[A] + 1) return false;
  const double kGeV = 2.99792458e-3, kPi = 3.14159265358979323846;
  const double Rm = p.pt_min / (kGeV * p.b_tesla);
  // B1
  const double r_lo = g.rho[A] - g.gap[A] / 2;
  const double r_hi = hypot(g.rho[A] + g.gap[A] / 2, g.hw[A]);
  const double rp_lo = g.rho[B] - g.gap[B] / 2;
  const double rp_hi = hypot(g.rho[B] + g.gap[B] / 2, g.hw[B]);
  // B2
  const double a_out = asin(fmin(1.0, rp_hi / (2 * Rm)));
  const double a_in = asin(fmin(1.0, r_lo / (2 * Rm)));
  // B3
  const double tol = atan(g.hw[A] / r_lo) + atan(g.hw[B] / rp_lo) + (a_out - a_in) + p.pad_phi;
  double d = fmod(g.phi[B] - g.phi[A], 2 * kPi);
  if (d > kPi) d -= 2 * kPi;
  if (d <= -kPi) d += 2 * kPi;
  if (!(fabs(d) <= tol)) return false;
  // B4
  const double ratio[2] = {rp_lo / r_hi, a_out / a_in};
  double z_lo = 0.0, z_hi = 0.0;
  bool first = true;
#pragma unroll
  for (int iz0 = 0; iz0 < 2; ++iz0)
#pragma unroll
    for (int iza = 0; iza < 2; ++iza)
#pragma unroll
      for (int ir = 0; ir < 2; ++ir) {
        const double z0 = iz0 ? p.z0_max : -p.z0_max;
        const double za = iza ? g.zhi[A] + p.pad_z : g.zlo[A] - p.pad_z;
        const double zp = z0 + (za - z0) * ratio[ir];
        if (first || zp < z_lo) z_lo = zp;
        if (first || zp > z_hi) z_hi = zp;
        first = false;
      }
  return z_hi >= g.zlo[B] && z_lo <= g.zhi[B];
}

// FILL = false: counts[A] = row length.  FILL = true: targets[offsets[A] ...] = the row, ascending.
template <bool FILL>
__global__ void __launch_bounds__(256) k_map_rows(const MapGeom g, const lst_map_params p, int* counts, const int* offsets,
                                                  int* targets) {
  __shared__ int s_warp[8];
  __shared__ int s_base;
  const int A = blockIdx.x;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (threadIdx.x == 0) s_base = FILL ? offsets[A] : 0;
  __syncthreads();
  for (int b0 = 0; b0 < g.n; b0 += 256) {
    const int B = b0 + threadIdx.x;
    const bool c = B < g.n && connected(g, p, A, B);
    const unsigned bal = __ballot_sync(0xffffffffu, c);
    if (lane == 0) s_warp[w] = __popc(bal);
    __syncthreads();
    int before = s_base, total = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      before += (i < w) ? s_warp[i] : 0;
      total += s_warp[i];
    }
    if (FILL && c) targets[before + __popc(bal & ((1u << lane) - 1u))] = B;
    __syncthreads();
    if (threadIdx.x == 0) s_base += total;
    __syncthreads();
  }
  if (!FILL && threadIdx.x == 0) counts[A] = s_base;
}

struct DeviceBuf {
  void* p = nullptr;
  ~DeviceBuf() { if (p) cudaFree(p); }
  cudaError_t alloc(size_t bytes) { return cudaMalloc(&p, bytes ? bytes : 1); }
};

}  // namespace

extern "C" int lst_build_module_map(const lst_map_geometry* mg, const lst_map_params* params, int device, int32_t* row_offsets,
                                    int32_t* targets, int64_t cap_targets, int64_t* n_targets, float* kernel_ms) {
  if (!mg || !row_offsets || !n_targets || mg->n_modules <= 0 || mg->n_modules > (1 << 24)) return LST_ERR_ARG;
  if (!mg->layer || !mg->phi || !mg->rho || !mg->gap || !mg->half_width || !mg->z_lo || !mg->z_hi) return LST_ERR_ARG;
  lst_map_params p;
  if (params) p = *params; else lst_default_map_params(&p);
  if (!(p.pt_min > 0.0) || !(p.b_tesla > 0.0) || !(p.z0_max >= 0.0)) return LST_ERR_ARG;
  const int n = mg->n_modules;
  for (int i = 0; i < n; ++i)
    if (mg->layer[i] < 0 || mg->layer[i] >= LST_N_LAYERS || !(mg->rho[i] - mg->gap[i] / 2 > 0.0) || !(mg->half_width[i] > 0.0)) return LST_ERR_ARG;
  *n_targets = 0;
  if (cudaSetDevice(device) != cudaSuccess) return LST_ERR_CUDA;
  DeviceBuf d_layer, d_f[6], d_counts, d_offsets, d_targets;
  const double* host_f[6] = {mg->phi, mg->rho, mg->gap, mg->half_width, mg->z_lo, mg->z_hi};
  if (d_layer.alloc(n) != cudaSuccess || d_counts.alloc(4 * (size_t)n) != cudaSuccess || d_offsets.alloc(4 * ((size_t)n + 1)) != cudaSuccess)
    return LST_ERR_NOMEM;
  if (cudaMemcpy(d_layer.p, mg->layer, n, cudaMemcpyHostToDevice) != cudaSuccess) return LST_ERR_CUDA;
  for (int k = 0; k < 6; ++k) {
    if (d_f[k].alloc(8 * (size_t)n) != cudaSuccess) return LST_ERR_NOMEM;
    if (cudaMemcpy(d_f[k].p, host_f[k], 8 * (size_t)n, cudaMemcpyHostToDevice) != cudaSuccess) return LST_ERR_CUDA;
  }
  MapGeom g{n, static_cast<const signed char*>(d_layer.p), static_cast<const double*>(d_f[0].p), static_cast<const double*>(d_f[1].p),
            static_cast<const double*>(d_f[2].p), static_cast<const double*>(d_f[3].p), static_cast<const double*>(d_f[4].p),
            static_cast<const double*>(d_f[5].p)};
  cudaEvent_t ev[4];
  for (auto& e : ev) cudaEventCreate(&e);
  cudaEventRecord(ev[0], 0);
  k_map_rows<false><<<n, 256>>>(g, p, static_cast<int*>(d_counts.p), nullptr, nullptr);
  cudaEventRecord(ev[1], 0);
  std::vector<int32_t> counts(n);
  int status = LST_OK;
  bool filled = false;
  if (cudaMemcpy(counts.data(), d_counts.p, 4 * (size_t)n, cudaMemcpyDeviceToHost) != cudaSuccess) status = LST_ERR_CUDA;
  int64_t total = 0;
  if (status == LST_OK) {
    for (int i = 0; i < n; ++i) { row_offsets[i] = (int32_t)total; total += counts[i]; }
    row_offsets[n] = (int32_t)total;
    *n_targets = total;                                   // on LST_ERR_OVERFLOW: the size the caller has to provide
    if (total > 0x7fffffffLL || total > cap_targets || (total > 0 && !targets)) status = LST_ERR_OVERFLOW;
  }
  if (status == LST_OK && total > 0) {
    if (d_targets.alloc(4 * (size_t)total) != cudaSuccess) status = LST_ERR_NOMEM;
    else if (cudaMemcpy(d_offsets.p, row_offsets, 4 * ((size_t)n + 1), cudaMemcpyHostToDevice) != cudaSuccess) status = LST_ERR_CUDA;
    else {
      cudaEventRecord(ev[2], 0);
      k_map_rows<true><<<n, 256>>>(g, p, nullptr, static_cast<const int*>(d_offsets.p), static_cast<int*>(d_targets.p));
      cudaEventRecord(ev[3], 0);
      filled = true;
      if (cudaMemcpy(targets, d_targets.p, 4 * (size_t)total, cudaMemcpyDeviceToHost) != cudaSuccess) status = LST_ERR_CUDA;
    }
  }
  if (cudaDeviceSynchronize() != cudaSuccess || cudaGetLastError() != cudaSuccess) status = status == LST_OK ? LST_ERR_CUDA : status;
  if (kernel_ms) {
    kernel_ms[0] = kernel_ms[1] = 0.0f;
    if (status != LST_ERR_CUDA) {
      cudaEventElapsedTime(&kernel_ms[0], ev[0], ev[1]);
      if (filled) cudaEventElapsedTime(&kernel_ms[1], ev[2], ev[3]);
    }
  }
  for (auto& e : ev) cudaEventDestroy(e);
  return status;
}

// ------------------------------------------------------------------------------------------
// lst_build_module_map_static: the same map without any allocation (include/lst.h).  Inputs and outputs are the caller's
// device arrays; the one piece of scratch -- the row lengths between the count pass and the scan -- is the file-scope array
// below.  In host code `g_map_row_len` is only a stand-in for the symbol: the kernels get the address that
// cudaGetSymbolAddress returns for the device that is current (looked up once per device, under a mutex).
// ------------------------------------------------------------------------------------------
namespace {

static __device__ __align__(256) int g_map_row_len[LST_MAP_STATIC_MAX_MODULES];

constexpr int kMaxDevices = 64;
std::mutex g_row_len_mu;
int* g_row_len_ptr[kMaxDevices] = {};

// `device` must be current.
cudaError_t row_len_scratch(int device, int** out) {
  std::lock_guard<std::mutex> lock(g_row_len_mu);
  if (!g_row_len_ptr[device]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_map_row_len);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_row_len_ptr[device] = static_cast<int*>(p);
  }
  *out = g_row_len_ptr[device];
  return cudaSuccess;
}

// k_map_rows with the fill bounded by the caller's buffer: FILL = false writes row_len[A]; FILL = true writes the entries of
// row A whose CSR position is below cap.
template <bool FILL>
__global__ void __launch_bounds__(256) k_map_rows_static(const MapGeom g, const lst_map_params p, int* row_len, const int* offsets,
                                                         int* targets, long long cap) {
  __shared__ int s_warp[8];
  __shared__ int s_base;
  const int A = blockIdx.x;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (threadIdx.x == 0) s_base = FILL ? offsets[A] : 0;
  __syncthreads();
  for (int b0 = 0; b0 < g.n; b0 += 256) {
    const int B = b0 + threadIdx.x;
    const bool c = B < g.n && connected(g, p, A, B);
    const unsigned bal = __ballot_sync(0xffffffffu, c);
    if (lane == 0) s_warp[w] = __popc(bal);
    __syncthreads();
    int before = s_base, total = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      before += (i < w) ? s_warp[i] : 0;
      total += s_warp[i];
    }
    if (FILL && c) {
      const int pos = before + __popc(bal & ((1u << lane) - 1u));
      if ((long long)pos < cap) targets[pos] = B;
    }
    __syncthreads();
    if (threadIdx.x == 0) s_base += total;
    __syncthreads();
  }
  if (!FILL && threadIdx.x == 0) row_len[A] = s_base;
}

// One block: offsets[i] = sum of row_len[0 .. i), offsets[n] = the number of connections (n <= 32768 rows of at most n
// entries: below 2^31).  1024 threads take 1024 rows per round and carry the running sum.
__global__ void __launch_bounds__(1024) k_map_scan_static(int n, const int* row_len, int* offsets) {
  __shared__ int s_warp[32];
  __shared__ int s_carry;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  if (tid == 0) s_carry = 0;
  __syncthreads();
  for (int i0 = 0; i0 < n; i0 += 1024) {
    const int i = i0 + tid;
    const int v = i < n ? row_len[i] : 0;
    int incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int u = __shfl_up_sync(0xffffffffu, incl, d);
      if (lane >= d) incl += u;
    }
    if (lane == 31) s_warp[w] = incl;
    __syncthreads();
    if (w == 0) {
      const int x = s_warp[lane];
      int xi = x;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const int u = __shfl_up_sync(0xffffffffu, xi, d);
        if (lane >= d) xi += u;
      }
      s_warp[lane] = xi - x;
    }
    __syncthreads();
    const int carry = s_carry;
    if (i < n) offsets[i] = carry + s_warp[w] + incl - v;
    __syncthreads();
    if (tid == 1023) s_carry = carry + s_warp[31] + incl;
    __syncthreads();
  }
  if (tid == 0) offsets[n] = s_carry;
}

}  // namespace

extern "C" int lst_build_module_map_static(const lst_map_geometry* mg, const lst_map_params* params, int device,
                                           int32_t* row_offsets, int32_t* targets, int64_t cap_targets, void* cuda_stream) {
  if (!mg || !row_offsets || mg->n_modules <= 0 || cap_targets < 0 || (cap_targets > 0 && !targets)) return LST_ERR_ARG;
  if (!mg->layer || !mg->phi || !mg->rho || !mg->gap || !mg->half_width || !mg->z_lo || !mg->z_hi) return LST_ERR_ARG;
  if (device < 0 || device >= kMaxDevices) return LST_ERR_ARG;
  lst_map_params p;
  if (params) p = *params; else lst_default_map_params(&p);
  if (!(p.pt_min > 0.0) || !(p.b_tesla > 0.0) || !(p.z0_max >= 0.0)) return LST_ERR_ARG;
  if (mg->n_modules > LST_MAP_STATIC_MAX_MODULES) return LST_ERR_LIMIT;   // the scratch array holds one int per module
  const int n = mg->n_modules;
  if (cudaSetDevice(device) != cudaSuccess) return LST_ERR_CUDA;
  int* row_len = nullptr;
  if (row_len_scratch(device, &row_len) != cudaSuccess) return LST_ERR_CUDA;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const MapGeom g{n, reinterpret_cast<const signed char*>(mg->layer), mg->phi, mg->rho, mg->gap, mg->half_width, mg->z_lo, mg->z_hi};
  // row_len[0 .. n) is written by the first kernel before the second reads it: nothing of the last call's contents is used
  k_map_rows_static<false><<<n, 256, 0, s>>>(g, p, row_len, nullptr, nullptr, 0);
  k_map_scan_static<<<1, 1024, 0, s>>>(n, row_len, row_offsets);
  k_map_rows_static<true><<<n, 256, 0, s>>>(g, p, nullptr, row_offsets, targets, (long long)cap_targets);
  return cudaGetLastError() == cudaSuccess ? LST_OK : LST_ERR_CUDA;
}

extern "C" int lst_default_map_params(lst_map_params* p) {
  if (!p) return LST_ERR_ARG;
  p->pt_min = 0.8;
  p->b_tesla = 3.8;
  p->z0_max = 15.0;
  p->pad_phi = 0.01;
  p->pad_z = 1.0;
  return LST_OK;
}
