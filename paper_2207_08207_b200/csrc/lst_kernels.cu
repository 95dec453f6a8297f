// lst_kernels.cu -- sm_100a kernels of the LST hot path (DESIGN.md sections 5-6).
//
// Hits and mini-doublets are kept ordered by azimuth inside their module, so the MD and the
// segment stage look only at a window of candidates found by binary search (DESIGN.md
// section 6); every candidate in a window goes through the exact SPEC selection.
//
// Every stage is  count -> (last block scans) -> fill : the count kernel evaluates the
// selection and leaves per-owner counts; the last block to finish turns block totals into block
// bases (no extra launch, no host round trip); the fill kernel re-walks the same candidates in
// the same order and writes each object at its final, deterministic position.  No global atomic
// is issued per candidate or per object: compaction is warp ballot + popc, block scan, and one
// ticket atomic per block.
//
// blockIdx.y = index of the event within the batch (lst_run_batch): all events of a batch go
// through one launch per kernel.
#include "lst_device.cuh"

namespace lst {

// ------------------------------------------------------------------------------------------
// small device utilities
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned lane_id() { return threadIdx.x & 31u; }
__device__ __forceinline__ unsigned lanemask_lt() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

__device__ __forceinline__ int warp_incl_scan(int v) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    int t = __shfl_up_sync(0xffffffffu, v, d);
    if ((int)lane_id() >= d) v += t;
  }
  return v;
}

// Exclusive scan of one int per thread over the block; returns the prefix, total in `total`.
// NT = blockDim.x (multiple of 32, <= 1024). Ends with a barrier: safe to call repeatedly.
template <int NT>
__device__ __forceinline__ int block_excl_scan(int v, int& total) {
  __shared__ int warp_sum[NT / 32];
  __shared__ int block_total;
  const int incl = warp_incl_scan(v);
  const int w = threadIdx.x >> 5;
  if (lane_id() == 31) warp_sum[w] = incl;
  __syncthreads();
  if (w == 0) {
    int s = (lane_id() < NT / 32) ? warp_sum[lane_id()] : 0;
    const int si = warp_incl_scan(s);
    if (lane_id() < NT / 32) warp_sum[lane_id()] = si - s;
    if (lane_id() == 31) block_total = si;
  }
  __syncthreads();
  const int r = incl - v + warp_sum[w];
  total = block_total;
  __syncthreads();
  return r;
}

// In-place exclusive scan of a[0..n) by the whole block, a[n] = total (unclamped total is
// returned to every thread). Values are read with ld.cg: they were written by other blocks.
// If clamp >= 0 the stored prefixes are min(prefix, clamp).
template <int NT>
__device__ int block_scan_array(int* a, int n, int clamp) {
  const int ipt = (n + NT - 1) / NT;
  const int lo = min(n, (int)threadIdx.x * ipt), hi = min(n, lo + ipt);
  int s = 0;
  for (int i = lo; i < hi; ++i) s += __ldcg(a + i);
  int total;
  int run = block_excl_scan<NT>(s, total);
  for (int i = lo; i < hi; ++i) {
    const int v = __ldcg(a + i);
    a[i] = (clamp >= 0) ? min(run, clamp) : run;
    run += v;
  }
  if (threadIdx.x == 0) a[n] = (clamp >= 0) ? min(total, clamp) : total;
  return total;
}

// In-place exclusive scan of the ints a[0 .. n] (a[n] must be 0 on entry and receives the total)
// by the whole block, 16 bytes per lane and coalesced.  The array is padded with zeros to a
// multiple of 4 ints (the slot layout rounds every array up to 256 bytes).  The values were
// written by other blocks: ld.cg.  Returns the total.
template <int NT>
__device__ int block_scan_array4(int* a, int n) {
  __shared__ int warp_tot[NT / 32];
  constexpr int W = NT / 32;
  int4* a4 = reinterpret_cast<int4*>(a);
  const int n4 = (n + 1 + 3) / 4, per = (n4 + W - 1) / W;
  const int w = threadIdx.x >> 5, lane = (int)lane_id();
  const int lo = min(n4, w * per), hi = min(n4, lo + per);
  int s = 0;
  for (int j = lo + lane; j < hi; j += 32) {
    const int4 v = __ldcg(a4 + j);
    s += (v.x + v.y) + (v.z + v.w);
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
  if (lane == 0) warp_tot[w] = s;
  __syncthreads();
  int carry = 0, total = 0;
#pragma unroll
  for (int i = 0; i < W; ++i) {
    const int v = warp_tot[i];
    carry += (i < w) ? v : 0;
    total += v;
  }
  for (int j0 = lo; j0 < hi; j0 += 32) {
    const int j = j0 + lane;
    int4 v = make_int4(0, 0, 0, 0);
    if (j < hi) v = __ldcg(a4 + j);
    const int t = (v.x + v.y) + (v.z + v.w);
    const int incl = warp_incl_scan(t);
    const int ex = carry + incl - t;
    if (j < hi) a4[j] = make_int4(ex, ex + v.x, ex + v.x + v.y, ex + v.x + v.y + v.z);
    carry += __shfl_sync(0xffffffffu, incl, 31);
  }
  __syncthreads();
  return total;
}

// Ticket: true in every thread of the block that finishes last among `n_blocks`.
__device__ __forceinline__ bool last_block_done(unsigned* counter, unsigned n_blocks) {
  __shared__ bool is_last;
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) {
    const unsigned t = atomicAdd(counter, 1u);
    is_last = (t == n_blocks - 1);
    if (is_last) atomicExch(counter, 0u);
  }
  __syncthreads();
  const bool r = is_last;
  if (r) __threadfence();
  return r;
}

__device__ __forceinline__ void publish_total(SlotHeader* h, int kind, int total, int cap) {
  h->needed[kind] = (unsigned long long)total;
  h->n[kind] = min(total, cap);
  if (total > cap) atomicOr(&h->overflow, 1 << kind);
}

// ------------------------------------------------------------------------------------------
// search windows.  A window is a conservative superset of what the SPEC
// selection can accept, derived from the selection's own inequalities and the per-event range
// of r per (side, layer); every candidate inside it goes through the exact SPEC selection, so
// the object set does not depend on the window.  Geometry of a pair seen from the beam line:
// with alpha the angle between the inner position vector and the inner->outer displacement
// (sin alpha is the cut variable sinA / sinS) and delta the azimuth difference,
//     delta = alpha - asin((r_in / r_out) sin alpha)          (law of sines; dot > 0, r_out > r_in)
// which grows with alpha, and for alpha > 0 with r_out.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ float delta_of(float s, float ratio) {
  return asinf(s) - asinf(ratio * s);
}

__device__ __forceinline__ int lower_bound_f(const float* a, int lo, int hi, float v) {  // first a[i] >= v
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (a[mid] < v) lo = mid + 1; else hi = mid;
  }
  return lo;
}
__device__ __forceinline__ int upper_bound_f(const float* a, int lo, int hi, float v) {  // first a[i] > v
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (a[mid] <= v) lo = mid + 1; else hi = mid;
  }
  return lo;
}

// M2 bounds |sinA| by thr(r_u) <= thr(r_max_upper); M1 (dot > 0) gives r_u > r_l.
// Returns the half width of the azimuth window around the lower hit, < 0 if nothing can pass.
__device__ __forceinline__ float md_window(const Cuts& c, int layer, float r_l, float r_max_upper) {
  if (!(r_max_upper > 0.0f) || !(r_max_upper * 1.000001f >= r_l)) return -1.0f;
  const float thr = fminf(1.0f, sin_threshold(c, r_max_upper, c.md_cos_eps[layer], c.md_sin_eps[layer]) * 1.00001f);
  const float d = delta_of(thr, fminf(1.0f, r_l / r_max_upper));
  return d * 1.001f + 2e-5f;
}

// S2 bounds |sinS| by thr(r_o); S4 on the inner MD bounds sinS * (ur_i / r_o) by sinA_i +- eps;
// S3 needs r_o > r_i.  [r_min_o, r_max_o] is the range of r of the anchors of the outer layer.
// Returns the window [dlo, dhi] of azimuth(outer) - azimuth(inner); dlo > dhi if nothing can pass.
__device__ __forceinline__ void seg_window(const Cuts& c, int layer, float r_i, float ur_i, float sinA_i,
                                           float r_min_o, float r_max_o, float& dlo, float& dhi) {
  dlo = 1.0f;
  dhi = -1.0f;
  if (!(r_max_o > r_i)) return;
  const float r_lo = fmaxf(r_min_o, r_i);
  float s_hi = fminf(1.0f, sin_threshold(c, r_max_o, c.seg_cos_eps, c.seg_sin_eps) * 1.00001f);
  float s_lo = -s_hi;
  if (ur_i > 0.0f && ur_i < 3.0e38f) {
    const float e = c.md_eps[layer] + 1e-5f;
    const float c_lo = (sinA_i - e) / ur_i, c_hi = (sinA_i + e) / ur_i;
    const float a = (c_lo >= 0.0f) ? c_lo * r_lo : c_lo * r_max_o;   // min over r_o of c_lo * r_o
    const float b = (c_hi >= 0.0f) ? c_hi * r_max_o : c_hi * r_lo;   // max over r_o of c_hi * r_o
    s_lo = fmaxf(s_lo, a - (1e-5f + 1e-5f * fabsf(a)));
    s_hi = fminf(s_hi, b + (1e-5f + 1e-5f * fabsf(b)));
  }
  if (!(s_lo <= s_hi)) return;
  const float q_lo = fminf(1.0f, r_i / r_lo), q_hi = r_i / r_max_o;
  const float hi = fmaxf(delta_of(s_hi, q_lo), delta_of(s_hi, q_hi));
  const float lo = fminf(delta_of(s_lo, q_lo), delta_of(s_lo, q_hi));
  dlo = lo - (3e-5f + 1e-3f * fabsf(lo));
  dhi = hi + (3e-5f + 1e-3f * fabsf(hi));
}

__device__ __forceinline__ float r_min_of(const SlotHeader* h, int side, int layer) {
  return __int_as_float(0x7f800000 - h->r_min_inv[side][layer]);
}
__device__ __forceinline__ float r_max_of(const SlotHeader* h, int side, int layer) {
  return __int_as_float(h->r_max[side][layer]);
}

// ------------------------------------------------------------------------------------------
// a0: load + bin by (side, module) + order by azimuth + derive r
// blockIdx.y = event of the batch; its input arrays come from the pointer table `B`.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_bin_count(const __grid_constant__ Params P, const __grid_constant__ HitBatch B) {
  Slot S(P, blockIdx.y);
  const HitInput& in = B.ev[blockIdx.y];
  unsigned* cnt = S.bin_start();
  const int nmod = P.L.n_modules;
  int bad = 0;
  for (int h = blockIdx.x * blockDim.x + threadIdx.x; h < in.n; h += gridDim.x * blockDim.x) {
    const int m = in.module[h];
    const unsigned sd = in.side[h];
    if (m < 0 || m >= nmod || sd > 1u) { ++bad; continue; }
    atomicAdd(cnt + ((int)sd * nmod + m), 1u);
  }
  if (bad) atomicAdd(&S.hdr()->bad_hits, bad);
  // the last block of the event turns the counts into bin offsets
  if (!last_block_done(&S.hdr()->done[4], gridDim.x)) return;
  int* start = reinterpret_cast<int*>(cnt);
  // search space of the MD stage: sum over modules of (#lower hits) x (#upper hits)
  unsigned long long c = 0;
#pragma unroll 4
  for (int m = threadIdx.x; m < nmod; m += 256)
    c += (unsigned long long)__ldcg(start + m) * (unsigned long long)__ldcg(start + nmod + m);
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) c += __shfl_down_sync(0xffffffffu, c, d);
  if (lane_id() == 0 && c) atomicAdd(&S.hdr()->cand[LST_MD_], c);
  __syncthreads();
  const int total = block_scan_array4<256>(start, P.L.n_bins);
  if (threadIdx.x == 0) {
    S.hdr()->n_hits = total;
    S.hdr()->n_lower = start[nmod];
  }
}

__global__ void __launch_bounds__(256) k_bin_scatter(const __grid_constant__ Params P, const __grid_constant__ HitBatch B) {
  Slot S(P, blockIdx.y);
  const HitInput& in = B.ev[blockIdx.y];
  const unsigned* start = S.bin_start();
  unsigned* cur = S.bin_cursor();
  int* tmp = S.tmp_idx();
  float* tkey = S.tmp_key();
  const int nmod = P.L.n_modules;
  for (int h = blockIdx.x * blockDim.x + threadIdx.x; h < in.n; h += gridDim.x * blockDim.x) {
    const int m = in.module[h];
    const unsigned sd = in.side[h];
    if (m < 0 || m >= nmod || sd > 1u) continue;
    const int b = (int)sd * nmod + m;
    const float x = in.x[h], y = in.y[h];
    const float2 cs = P.mod_cs[m];
    // azimuth relative to the module normal; non-finite hits (they can never pass a cut) go last
    const float k = atan2f(cs.x * y - cs.y * x, cs.x * x + cs.y * y);
    const unsigned pos = start[b] + atomicAdd(cur + b, 1u);
    tmp[pos] = h;
    tkey[pos] = (fabsf(k) <= 4.0f) ? k : 3.0e38f;
  }
}

// One warp per bin: order the bin's hits by (key, original index) and gather the coordinates.
// n <= 32: rank by shuffles; n <= kSortMax: bitonic sort of 64-bit (key, index) words in shared
// memory; beyond: rank by an O(n^2) sweep over global memory.
constexpr int kSortMax = 256;
constexpr int kOrderWarps = 8;

__device__ __forceinline__ unsigned ordered_bits(float f) {  // monotone map float -> unsigned
  const unsigned u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

__global__ void __launch_bounds__(kOrderWarps * 32) k_bin_order(const __grid_constant__ Params P, const __grid_constant__ HitBatch B) {
  __shared__ unsigned long long sortbuf[kOrderWarps][kSortMax];
  Slot S(P, blockIdx.y);
  const HitInput& in = B.ev[blockIdx.y];
  const int wib = threadIdx.x >> 5, lane = (int)lane_id();
  const int b = blockIdx.x * kOrderWarps + wib;
  if (b >= P.L.n_bins) return;
  const unsigned* start = S.bin_start();
  const int s = start[b], n = start[b + 1] - s;
  if (n == 0) return;
  const int nmod = P.L.n_modules;
  const int side = b >= nmod, m = b - side * nmod;
  const int* tmp = S.tmp_idx() + s;
  const float* tkey = S.tmp_key() + s;
  float4* hit4 = S.hit4() + s;
  float* hkey = S.hit_key() + s;
  int* orig = S.hit_orig() + s;
  int* hmod = S.hit_module() + s;
  float rmin = 3.0e38f, rmax = 0.0f;
  unsigned long long* buf = sortbuf[wib];
  const bool sorted = n > 32 && n <= kSortMax;
  if (sorted) {
    int N = 64;
    while (N < n) N <<= 1;
    for (int i = lane; i < N; i += 32)
      buf[i] = (i < n) ? (((unsigned long long)ordered_bits(tkey[i]) << 32) | (unsigned)tmp[i]) : ~0ull;
    __syncwarp();
    for (int k = 2; k <= N; k <<= 1) {
      for (int j = k >> 1; j > 0; j >>= 1) {
        for (int p = lane; p < (N >> 1); p += 32) {
          const int i = ((p & ~(j - 1)) << 1) | (p & (j - 1)), l = i | j;
          const unsigned long long a = buf[i], c = buf[l];
          const bool up = (i & k) == 0;
          if ((a > c) == up) { buf[i] = c; buf[l] = a; }
        }
        __syncwarp();
      }
    }
  }
  for (int i0 = 0; i0 < n; i0 += 32) {
    const int i = i0 + lane;
    int mine = 0, rank = i;
    float key = 0.0f;
    if (sorted) {
      if (i < n) {
        mine = (int)(unsigned)(buf[i] & 0xffffffffull);
        const unsigned u = (unsigned)(buf[i] >> 32);
        key = __uint_as_float((u & 0x80000000u) ? (u & 0x7fffffffu) : ~u);
      }
    } else {
      if (i < n) { mine = tmp[i]; key = tkey[i]; }
      rank = 0;
      if (n <= 32) {
        for (int j = 0; j < n; ++j) {
          const float kj = __shfl_sync(0xffffffffu, key, j);
          const int ij = __shfl_sync(0xffffffffu, mine, j);
          rank += (kj < key) || (kj == key && ij < mine);
        }
      } else if (i < n) {
        for (int j = 0; j < n; ++j) {
          const float kj = tkey[j];
          const int ij = tmp[j];
          rank += (kj < key) || (kj == key && ij < mine);
        }
      }
    }
    if (i < n) {
      const float x = in.x[mine], y = in.y[mine], z = in.z[mine];
      const float r = sqrtf(x * x + y * y);
      hit4[rank] = make_float4(x, y, z, r);
      hkey[rank] = key;
      orig[rank] = mine;
      hmod[rank] = m;
      if (r < 3.0e38f) { rmin = fminf(rmin, r); rmax = fmaxf(rmax, r); }
    }
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    rmin = fminf(rmin, __shfl_down_sync(0xffffffffu, rmin, d));
    rmax = fmaxf(rmax, __shfl_down_sync(0xffffffffu, rmax, d));
  }
  if (lane == 0 && rmin <= rmax) {
    const int layer = P.mod_layer[m];
    SlotHeader* h = S.hdr();
    atomicMax(&h->r_min_inv[side][layer], 0x7f800000 - __float_as_int(rmin));
    atomicMax(&h->r_max[side][layer], __float_as_int(rmax));
  }
}

// ------------------------------------------------------------------------------------------
// a1: mini-doublets. One thread per lower hit; its candidates are the upper hits of the same
// module inside the azimuth window (a binary search in the key-ordered upper bin).
// ------------------------------------------------------------------------------------------
template <bool FILL>
__global__ void __launch_bounds__(kScanChunk) k_md(const __grid_constant__ Params P) {
  Slot S(P, blockIdx.y);
  SlotHeader* H = S.hdr();
  const int nmod = P.L.n_modules;
  const int nLower = H->n_lower;
  const int nChunks = (nLower + kScanChunk - 1) / kScanChunk;
  const unsigned* bs = S.bin_start();
  const float4* hit4 = S.hit4();
  const float* hkey = S.hit_key();
  int* md_off = S.md_off();
  int* block_base = S.md_block_base();
  unsigned long long evals = 0;
  for (int c = blockIdx.x; c < nChunks; c += gridDim.x) {
    const int i = c * kScanChunk + threadIdx.x;
    int count = 0;
    if (i < nLower) {
      const int m = S.hit_module()[i];
      const int layer = P.mod_layer[m];
      const int u0 = bs[nmod + m], u1 = bs[nmod + m + 1];
      if (u1 > u0) {
        const float4 lo = hit4[i];
        const float kl = hkey[i];
        const float w = md_window(P.cuts, layer, lo.w, r_max_of(H, 1, layer));
        int j0 = u0, j1 = u1;
        if (w < 0.0f) {
          j1 = j0;
        } else if (fabsf(kl) + w < 1.5f) {
          j0 = lower_bound_f(hkey, u0, u1, kl - w);
          j1 = upper_bound_f(hkey, j0, u1, kl + w);
        }
        evals += (unsigned long long)(j1 - j0);
        const int base = FILL ? block_base[c] + md_off[i] : 0;
        for (int j = j0; j < j1; ++j) {
          const float4 up = hit4[j];
          MdOut o;
          if (md_select(P.cuts, layer, lo, up, o)) {
            if (FILL) {
              const int pos = base + count;
              if (pos < P.L.cap_md) {
                S.md_anchor()[pos] = lo;
                S.md_aux()[pos] = make_float2(up.w, o.sinA);
                S.md_key()[pos] = kl;
                S.md_hits()[pos] = make_int2(S.hit_orig()[i], S.hit_orig()[j]);
                S.md_out()[pos] = make_float2(atan2f(lo.x * up.y - lo.y * up.x, lo.x * up.x + lo.y * up.y),
                                              atan2f(o.cross, o.dot));
                S.md_module()[pos] = m;
              }
            }
            ++count;
          }
        }
      }
    }
    if (!FILL) {
      int tot;
      const int ex = block_excl_scan<kScanChunk>(count, tot);
      if (i < nLower) md_off[i] = ex;
      if (threadIdx.x == 0) block_base[c] = tot;
    }
  }
  if (FILL) {
    // md_start[m] = index of the first MD of module m = offset of the module's first lower hit
    const int total = H->n[LST_MD_];
    for (int m = blockIdx.x * kScanChunk + threadIdx.x; m <= nmod; m += gridDim.x * kScanChunk) {
      const int ls = (m < nmod) ? (int)bs[m] : nLower;
      const int b0 = (ls < nLower) ? min(block_base[ls / kScanChunk] + md_off[ls], P.L.cap_md) : total;
      S.md_start()[m] = b0;
      if (m < nmod) {
        // (first MD, end MD, key range of the module's lower hits >= key range of its MDs)
        const int le = (int)bs[m + 1];
        const int b1 = (le < nLower) ? min(block_base[le / kScanChunk] + md_off[le], P.L.cap_md) : total;
        const bool any = le > ls;
        S.mod_info()[m] = make_int4(b0, b1, __float_as_int(any ? hkey[ls] : 3.0e38f), __float_as_int(any ? hkey[le - 1] : -3.0e38f));
      }
    }
  } else {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) evals += __shfl_down_sync(0xffffffffu, evals, d);
    if (lane_id() == 0 && evals) atomicAdd(&H->eval[LST_MD_], evals);
    if (last_block_done(&H->done[0], gridDim.x)) {
      const int total = block_scan_array<kScanChunk>(block_base, nChunks, -1);
      if (threadIdx.x == 0) publish_total(H, LST_MD_, total, P.L.cap_md);
    }
  }
}

// ------------------------------------------------------------------------------------------
// single-pass ordered output: chunks of owners are handed out in order by a ticket; a block
// learns where its chunk's objects start by decoupled look-back over the totals of the chunks
// before it (each chunk publishes its total as soon as it is known, so nothing waits on a
// block that has not started).  status word: bits 63:62 = 1 total only, 2 = inclusive prefix.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void st_status(unsigned long long* p, unsigned long long v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_status(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
// Called by all lanes of ONE warp. Returns the number of objects of chunks 0 .. c-1.
__device__ __forceinline__ int lookback_exclusive(unsigned long long* status, int c, int total) {
  const int lane = (int)lane_id();
  if (lane == 0) st_status(status + c, ((c == 0 ? 2ull : 1ull) << 62) | (unsigned)total);
  if (c == 0) return 0;
  int sum = 0;
  for (int j = c - 1;; j -= 32) {
    const int idx = j - lane;
    unsigned long long v = (idx >= 0) ? ld_status(status + idx) : (2ull << 62);
    while (__any_sync(0xffffffffu, (v >> 62) == 0)) {
      if ((v >> 62) == 0) v = ld_status(status + idx);
    }
    const unsigned pmask = __ballot_sync(0xffffffffu, (v >> 62) == 2);
    const int firstP = pmask ? __ffs(pmask) - 1 : 32;
    int contrib = (lane <= firstP) ? (int)(unsigned)(v & 0xffffffffull) : 0;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) contrib += __shfl_xor_sync(0xffffffffu, contrib, d);
    sum += contrib;
    if (pmask) break;
  }
  if (lane == 0) st_status(status + c, (2ull << 62) | (unsigned)(sum + total));
  return sum;
}

// Exclusive max-scan of one non-negative int per thread over the block (0 for thread 0).
// Ends with a barrier.
template <int NT>
__device__ __forceinline__ int block_excl_scan_max(int v) {
  __shared__ int warp_max[NT / 32];
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int t = __shfl_up_sync(0xffffffffu, v, d);
    if ((int)lane_id() >= d) v = max(v, t);
  }
  const int w = threadIdx.x >> 5;
  if (lane_id() == 31) warp_max[w] = v;
  int ex = __shfl_up_sync(0xffffffffu, v, 1);
  if (lane_id() == 0) ex = 0;
  __syncthreads();
#pragma unroll
  for (int i = 0; i < NT / 32; ++i) ex = (i < w) ? max(ex, warp_max[i]) : ex;
  __syncthreads();
  return ex;
}

// ------------------------------------------------------------------------------------------
// a2: segments, single pass. One block per chunk of kSegChunk consecutive inner MDs (they may
// sit in several modules).  (1) every (inner MD, connected module) pair finds its window of
// outer MDs by a binary search in the connected module's key-ordered MD list, (2) a block scan
// of the window sizes numbers the candidates in (inner MD, outer MD) order, (3) one thread per
// candidate evaluates the SPEC selection ONCE; what passes is kept in shared memory, in order,
// until the look-back has told the block where its segments start.  Segments come out ordered
// by (inner MD, outer MD).
// ------------------------------------------------------------------------------------------
constexpr int kSegThreads = 128;
constexpr int kSegChunk = kSegChunkMd;  // inner MDs per chunk
constexpr int kSegPairs = 1024;  // (inner MD, connected module) pairs per tile (>= kMaxRow)
constexpr int kSegCand = 1024;   // candidates per lookup tile
constexpr int kSegStash = 512;   // segments of a chunk kept in shared memory

struct SegShared {
  float4 iAnchor[kSegChunk];
  float2 iAux[kSegChunk];
  float iKey[kSegChunk], iDlo[kSegChunk], iDhi[kSegChunk];
  int iRow0[kSegChunk], iNt[kSegChunk], iLayer[kSegChunk], kCnt[kSegChunk];
  int pLo[kSegPairs], pOff[kSegPairs + 1];
  unsigned short cPair[kSegCand];
  int stKO[kSegStash];
  float4 stV[kSegStash];
  int warpTot[kSegThreads / 32];
  float rMinO[6], rMaxO[6];
  int chunk, base, tMax;
};

// Walks the chunk's candidates in order. direct = false: passing candidates go to the stash
// (positions < kSegStash) and are counted per inner MD; direct = true: they are written to
// global memory at `base` + position.  Returns the number of passing candidates.
__device__ __forceinline__ int seg_walk(const Params& P, const Slot& S, SegShared& sh, int i0, int kn, int tStar,
                                        bool direct, int base, unsigned long long& space, unsigned long long& evals) {
  const float4* anchor = S.md_anchor();
  const float2* aux = S.md_aux();
  const float* mkey = S.md_key();
  const int4* mod_info = S.mod_info();
  const int tid = threadIdx.x, warp = tid >> 5;
  const unsigned magic = 0xffffffffu / (unsigned)tStar + 1u;  // q / tStar == umulhi(q, magic) for q < 65536
  const int kTile = min(kn, kSegPairs / tStar);
  int running = 0;  // passing candidates so far (uniform across the block)
  for (int kb = 0; kb < kn; kb += kTile) {
    const int kt = min(kTile, kn - kb), nPairs = kt * tStar;
    // (1) windows
    for (int q = tid; q < nPairs; q += kSegThreads) {
      const int kk = (int)__umulhi((unsigned)q, magic), t = q - kk * tStar, k = kb + kk;
      int first = 0, n = 0;
      if (t < sh.iNt[k]) {
        const int e = sh.iRow0[k] + t;
        const int4 info = mod_info[P.map_targets[e]];
        const int b0 = info.x, b1 = info.y;
        if (!direct) space += (unsigned long long)(b1 - b0);
        const float dlo = sh.iDlo[k], dhi = sh.iDhi[k];
        if (b1 > b0 && dlo <= dhi) {
          const float c0 = sh.iKey[k] + P.map_dphi[e];
          if (!(fabsf(c0) + fmaxf(fabsf(dlo), fabsf(dhi)) < 3.0f)) {
            first = b0;  // azimuth wrap possible (never with a sane geometry): no window
            n = b1 - b0;
          } else if (c0 + dhi >= __int_as_float(info.z) && c0 + dlo <= __int_as_float(info.w)) {
            first = lower_bound_f(mkey, b0, b1, c0 + dlo);
            n = upper_bound_f(mkey, first, b1, c0 + dhi) - first;
          }
        }
      }
      sh.pLo[q] = first;
      sh.pOff[q] = n;
    }
    __syncthreads();
    // (2) exclusive scan of the window sizes
    int nCand;
    {
      const int ipt = (nPairs + kSegThreads - 1) / kSegThreads;
      const int lo = min(nPairs, tid * ipt), hi = min(nPairs, lo + ipt);
      int s = 0;
      for (int q = lo; q < hi; ++q) s += sh.pOff[q];
      int run = block_excl_scan<kSegThreads>(s, nCand);
      for (int q = lo; q < hi; ++q) {
        const int v = sh.pOff[q];
        sh.pOff[q] = run;
        run += v;
      }
      if (tid == 0) sh.pOff[nPairs] = nCand;
    }
    __syncthreads();
    if (!direct && tid == 0) evals += (unsigned long long)nCand;
    for (int cb = 0; cb < nCand; cb += kSegCand) {
      const int nc = min(kSegCand, nCand - cb);
      // candidate -> pair table: every non-empty pair marks its first candidate, a max-scan fills the rest
      for (int j = tid; j < nc; j += kSegThreads) sh.cPair[j] = 0;
      __syncthreads();
      for (int q = tid; q < nPairs; q += kSegThreads) {
        const int s = sh.pOff[q];
        if (sh.pOff[q + 1] > s && s >= cb && s < cb + nc) sh.cPair[s - cb] = (unsigned short)q;
      }
      if (tid == 0 && cb > 0) {
        int lo = 0, hi = nPairs;  // last q with pOff[q] <= cb: the pair candidate cb belongs to
        while (hi - lo > 1) {
          const int mid = (lo + hi) >> 1;
          if (sh.pOff[mid] <= cb) lo = mid; else hi = mid;
        }
        sh.cPair[0] = (unsigned short)lo;
      }
      __syncthreads();
      {
        const int ipt = (nc + kSegThreads - 1) / kSegThreads;
        const int lo = min(nc, tid * ipt), hi = min(nc, lo + ipt);
        int m = 0;
        for (int j = lo; j < hi; ++j) m = max(m, (int)sh.cPair[j]);
        int carry = block_excl_scan_max<kSegThreads>(m);  // max over the entries of the threads before
        for (int j = lo; j < hi; ++j) {
          carry = max(carry, (int)sh.cPair[j]);
          sh.cPair[j] = (unsigned short)carry;
        }
      }
      __syncthreads();
      // (3) one thread per candidate
      for (int j0 = 0; j0 < nc; j0 += kSegThreads) {
        const int j = j0 + tid;
        bool pass = false;
        SegOut so;
        int k = 0, o = 0;
        if (j < nc) {
          const int q = sh.cPair[j];
          k = kb + (int)__umulhi((unsigned)q, magic);
          o = sh.pLo[q] + (cb + j - sh.pOff[q]);
          pass = seg_select(P.cuts, sh.iLayer[k], sh.iAnchor[k], sh.iAux[k], anchor[o], aux[o], so);
        }
        const unsigned bal = __ballot_sync(0xffffffffu, pass);
        if (lane_id() == 0) sh.warpTot[warp] = __popc(bal);
        __syncthreads();
        int before = 0, all = 0;
#pragma unroll
        for (int w = 0; w < kSegThreads / 32; ++w) {
          const int v = sh.warpTot[w];
          before += (w < warp) ? v : 0;
          all += v;
        }
        if (pass) {
          const int pos = running + before + __popc(bal & lanemask_lt());
          if (!direct) {
            atomicAdd(&sh.kCnt[k], 1);
            if (pos < kSegStash) {
              sh.stKO[pos] = (k << 24) | o;
              sh.stV[pos] = make_float4(so.sinS, so.z0, so.cross, so.dot);
            }
          } else if (base + pos < P.L.cap_seg) {
            const float4 ai = sh.iAnchor[k], ao = anchor[o];
            S.seg_md()[base + pos] = make_int2(i0 + k, o);
            S.seg_f()[base + pos] = make_float4(so.sinS, so.z0,
                                                atan2f(ai.x * ao.y - ai.y * ao.x, ai.x * ao.x + ai.y * ao.y),
                                                atan2f(so.cross, so.dot));
          }
        }
        running += all;
        __syncthreads();
      }
    }
    __syncthreads();
  }
  return running;
}

__global__ void __launch_bounds__(kSegThreads) k_seg(const __grid_constant__ Params P) {
  __shared__ SegShared sh;
  Slot S(P, blockIdx.y);
  SlotHeader* H = S.hdr();
  const int nMD = H->n[LST_MD_];
  const int nChunks = (nMD + kSegChunk - 1) / kSegChunk;
  int* seg_start = S.seg_start();
  const float4* anchor = S.md_anchor();
  const int tid = threadIdx.x;
  if (tid < 6) {
    sh.rMinO[tid] = r_min_of(H, 0, tid);
    sh.rMaxO[tid] = r_max_of(H, 0, tid);
  }
  unsigned long long space = 0, evals = 0;
  for (;;) {
    __syncthreads();  // previous chunk fully consumed (and rMinO / rMaxO visible)
    if (tid == 0) {
      sh.chunk = (int)atomicAdd(&H->ticket[LST_SEG_], 1u);
      sh.tMax = 0;
    }
    __syncthreads();
    const int c = sh.chunk;
    if (c >= nChunks) {
      if (c == 0 && tid == 0) {  // no MDs at all: the first ticket publishes the empty result
        publish_total(H, LST_SEG_, 0, P.L.cap_seg);
        seg_start[0] = 0;
      }
      break;
    }
    const int i0 = c * kSegChunk, kn = min(kSegChunk, nMD - i0);
    int nt = 0;
    if (tid < kn) {
      const int i = i0 + tid;
      const float4 a = anchor[i];
      const float2 x = S.md_aux()[i];
      const int A = S.md_module()[i];
      const int row0 = P.map_offsets[A];
      nt = P.map_offsets[A + 1] - row0;
      const int layer = P.mod_layer[A];
      float dlo = 1.0f, dhi = -1.0f;
      if (nt > 0) seg_window(P.cuts, layer, a.w, x.x, x.y, sh.rMinO[layer + 1], sh.rMaxO[layer + 1], dlo, dhi);
      sh.iAnchor[tid] = a;
      sh.iAux[tid] = x;
      sh.iKey[tid] = S.md_key()[i];
      sh.iDlo[tid] = dlo;
      sh.iDhi[tid] = dhi;
      sh.iRow0[tid] = row0;
      sh.iNt[tid] = nt;
      sh.iLayer[tid] = layer;
    }
    if (tid < kSegChunk) sh.kCnt[tid] = 0;
    if (tid < kSegChunk) {  // warps 0 and 1
      const int m = __reduce_max_sync(0xffffffffu, nt);
      if (lane_id() == 0 && m > 0) atomicMax(&sh.tMax, m);
    }
    __syncthreads();
    const int tStar = sh.tMax;
    int total = 0;
    if (tStar > 0) total = seg_walk(P, S, sh, i0, kn, tStar, false, 0, space, evals);
    // where do this chunk's segments start?
    if (tid < 32) {
      const int b = lookback_exclusive(S.lb_seg(), c, total);
      if (tid == 0) sh.base = b;
    }
    __syncthreads();
    const int base = sh.base;
    if (total <= kSegStash) {
      for (int j = tid; j < total; j += kSegThreads) {
        const int ko = sh.stKO[j], k = (int)((unsigned)ko >> 24), o = ko & 0xffffff;
        if (base + j < P.L.cap_seg) {
          const float4 v = sh.stV[j], ai = sh.iAnchor[k], ao = anchor[o];
          S.seg_md()[base + j] = make_int2(i0 + k, o);
          S.seg_f()[base + j] = make_float4(v.x, v.y, atan2f(ai.x * ao.y - ai.y * ao.x, ai.x * ao.x + ai.y * ao.y),
                                            atan2f(v.z, v.w));
        }
      }
    } else {
      seg_walk(P, S, sh, i0, kn, tStar, true, base, space, evals);  // rare: more segments than the stash holds
    }
    // first segment of every inner MD of the chunk
    {
      const int v = (tid < kn) ? sh.kCnt[tid] : 0;
      int tot;
      const int ex = block_excl_scan<kSegThreads>(v, tot);
      if (tid < kn) seg_start[i0 + tid] = min(base + ex, P.L.cap_seg);
    }
    if (c == nChunks - 1 && tid == 0) {
      publish_total(H, LST_SEG_, base + total, P.L.cap_seg);
      seg_start[nMD] = min(base + total, P.L.cap_seg);
    }
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) space += __shfl_down_sync(0xffffffffu, space, d);
  if (lane_id() == 0 && space) atomicAdd(&H->cand[LST_SEG_], space);
  if (tid == 0 && evals) atomicAdd(&H->eval[LST_SEG_], evals);
}

// ------------------------------------------------------------------------------------------
// a3: triplets. One thread per first segment a = (m1, m2); candidates are the segments leaving
// m2, a contiguous range because segments are stored by inner MD.
// ------------------------------------------------------------------------------------------
template <bool FILL>
__global__ void __launch_bounds__(kScanChunk) k_t3(const __grid_constant__ Params P) {
  Slot S(P, blockIdx.y);
  SlotHeader* H = S.hdr();
  const int nSeg = H->n[LST_SEG_];
  const int nChunks = (nSeg + kScanChunk - 1) / kScanChunk;
  const int* seg_start = S.seg_start();
  const int2* seg_md = S.seg_md();
  const float4* anchor = S.md_anchor();
  int* t3_start = S.t3_start();
  unsigned long long cand = 0;
  for (int c = blockIdx.x; c < nChunks; c += gridDim.x) {
    const int a = c * kScanChunk + threadIdx.x;
    int count = 0;
    if (a < nSeg) {
      const int2 ma = seg_md[a];
      const int b0 = seg_start[ma.y], b1 = seg_start[ma.y + 1];
      const float4 p1 = anchor[ma.x], p2 = anchor[ma.y];
      const int layer = P.mod_layer[S.md_module()[ma.x]];
      const int base = FILL ? S.t3_block_base()[c] + t3_start[a] : 0;
      cand += (unsigned long long)(b1 - b0);
      for (int b = b0; b < b1; ++b) {
        const int m3 = seg_md[b].y;
        float kappa, chi2;
        if (t3_select(P.cuts, layer, p1, p2, anchor[m3], kappa, chi2)) {
          if (FILL) {
            const int pos = base + count;
            if (pos < P.L.cap_t3) {
              S.t3_pack()[pos] = make_int4(ma.x, ma.y, m3, __float_as_int(kappa));
              S.t3_seg()[pos] = make_int2(a, b);
              S.t3_chi2()[pos] = chi2;
            }
          }
          ++count;
        }
      }
      if (FILL) t3_start[a] = min(base, P.L.cap_t3);
    }
    if (!FILL) {
      int tot;
      const int ex = block_excl_scan<kScanChunk>(count, tot);
      if (a < nSeg) t3_start[a] = ex;
      if (threadIdx.x == 0) S.t3_block_base()[c] = tot;
    }
  }
  if (!FILL) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) cand += __shfl_down_sync(0xffffffffu, cand, d);
    if (lane_id() == 0 && cand) { atomicAdd(&H->cand[LST_T3_], cand); atomicAdd(&H->eval[LST_T3_], cand); }
    if (last_block_done(&H->done[2], gridDim.x)) {
      const int total = block_scan_array<kScanChunk>(S.t3_block_base(), nChunks, -1);
      if (threadIdx.x == 0) {
        publish_total(H, LST_T3_, total, P.L.cap_t3);
        t3_start[nSeg] = min(total, P.L.cap_t3);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------
// a4: quintuplets. One thread per inner triplet A = (m1, m2, m3); candidates are the triplets
// whose first MD is m3: [t3_start[seg_start[m3]], t3_start[seg_start[m3 + 1]]), contiguous
// because triplets are stored by first segment and segments by inner MD.
// ------------------------------------------------------------------------------------------
template <bool FILL>
__global__ void __launch_bounds__(kScanChunk) k_t5(const __grid_constant__ Params P) {
  Slot S(P, blockIdx.y);
  SlotHeader* H = S.hdr();
  const int nT3 = H->n[LST_T3_];
  const int nChunks = (nT3 + kScanChunk - 1) / kScanChunk;
  const int* seg_start = S.seg_start();
  const int* t3_start = S.t3_start();
  const int4* t3_pack = S.t3_pack();
  const float4* anchor = S.md_anchor();
  int* t5_start = S.t5_start();
  unsigned long long cand = 0;
  for (int c = blockIdx.x; c < nChunks; c += gridDim.x) {
    const int A = c * kScanChunk + threadIdx.x;
    int count = 0;
    if (A < nT3) {
      const int4 ta = t3_pack[A];
      const int B0 = t3_start[seg_start[ta.z]], B1 = t3_start[seg_start[ta.z + 1]];
      const int base = FILL ? S.t5_block_base()[c] + t5_start[A] : 0;
      cand += (unsigned long long)(B1 - B0);
      if (B1 > B0) {
        float4 p[5];
        p[0] = anchor[ta.x];
        p[1] = anchor[ta.y];
        p[2] = anchor[ta.z];
        const int layer = P.mod_layer[S.md_module()[ta.x]];
        const float kA = __int_as_float(ta.w);
        for (int B = B0; B < B1; ++B) {
          const int4 tb = t3_pack[B];
          const float kB = __int_as_float(tb.w);
          p[3] = anchor[tb.y];
          p[4] = anchor[tb.z];
          T5Out o;
          if (layer <= 1 && t5_select(P.cuts, layer, kA, kB, p, o)) {
            if (FILL) {
              const int pos = base + count;
              if (pos < P.L.cap_t5) {
                int* md = S.t5_md() + 5 * (size_t)pos;
                md[0] = ta.x; md[1] = ta.y; md[2] = ta.z; md[3] = tb.y; md[4] = tb.z;
                S.t5_t3()[pos] = make_int2(A, B);
                float* f = S.t5_f() + 5 * (size_t)pos;
                f[0] = kA; f[1] = kB; f[2] = o.kfit; f[3] = o.chi2xy; f[4] = o.chi2rz;
              }
            }
            ++count;
          }
        }
      }
      if (FILL) t5_start[A] = min(base, P.L.cap_t5);
    }
    if (!FILL) {
      int tot;
      const int ex = block_excl_scan<kScanChunk>(count, tot);
      if (A < nT3) t5_start[A] = ex;
      if (threadIdx.x == 0) S.t5_block_base()[c] = tot;
    }
  }
  if (!FILL) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) cand += __shfl_down_sync(0xffffffffu, cand, d);
    if (lane_id() == 0 && cand) { atomicAdd(&H->cand[LST_T5_], cand); atomicAdd(&H->eval[LST_T5_], cand); }
    if (last_block_done(&H->done[3], gridDim.x)) {
      const int total = block_scan_array<kScanChunk>(S.t5_block_base(), nChunks, -1);
      if (threadIdx.x == 0) {
        publish_total(H, LST_T5_, total, P.L.cap_t5);
        t5_start[nT3] = min(total, P.L.cap_t5);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------
// output helpers: original-hit-index tuples and float payloads, one thread per object
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_gather_hits(const __grid_constant__ Params P, int kind, int n) {
  Slot S(P, 0);
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int2* mh = S.md_hits();
  int2* out = reinterpret_cast<int2*>(S.scratch());
  if (kind == LST_MD_) {
    out[i] = mh[i];
  } else if (kind == LST_SEG_) {
    const int2 s = S.seg_md()[i];
    out[2 * (size_t)i] = mh[s.x];
    out[2 * (size_t)i + 1] = mh[s.y];
  } else if (kind == LST_T3_) {
    const int4 t = S.t3_pack()[i];
    out[3 * (size_t)i] = mh[t.x];
    out[3 * (size_t)i + 1] = mh[t.y];
    out[3 * (size_t)i + 2] = mh[t.z];
  } else {
    const int* md = S.t5_md() + 5 * (size_t)i;
#pragma unroll
    for (int k = 0; k < 5; ++k) out[5 * (size_t)i + k] = mh[md[k]];
  }
}

__global__ void __launch_bounds__(256) k_pack_values(const __grid_constant__ Params P, int kind, int n) {
  Slot S(P, 0);
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float* out = reinterpret_cast<float*>(S.scratch());
  if (kind == LST_MD_) {
    const float2 o = S.md_out()[i];
    reinterpret_cast<float4*>(out)[i] = make_float4(S.md_aux()[i].y, o.x, o.y, S.md_anchor()[i].w);
  } else if (kind == LST_T3_) {
    reinterpret_cast<float2*>(out)[i] = make_float2(__int_as_float(S.t3_pack()[i].w), S.t3_chi2()[i]);
  }
}

// ------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------
// `ev` (optional, timing mode): ev[0] is recorded before the first kernel, ev[k + 1] after kernel k.
#define LST_EV(k) do { if (ev) cudaEventRecord(ev[k], s); } while (0)

int launch_bin(const Params& P, const HitBatch& in, int n_batch, cudaStream_t s, cudaEvent_t* ev) {
  int n_max = 0;
  for (int b = 0; b < n_batch; ++b) n_max = max(n_max, in.ev[b].n);
  const int per_event = max(8, 1184 / n_batch);
  const dim3 g(max(1, min((n_max + 255) / 256, per_event)), (unsigned)n_batch);
  LST_EV(0);
  k_bin_count<<<g, 256, 0, s>>>(P, in);   // + scan of the bin counts by the event's last block
  LST_EV(1);
  LST_EV(2);
  k_bin_scatter<<<g, 256, 0, s>>>(P, in);
  LST_EV(3);
  k_bin_order<<<dim3((P.L.n_bins + kOrderWarps - 1) / kOrderWarps, (unsigned)n_batch), kOrderWarps * 32, 0, s>>>(P, in);
  LST_EV(4);
  return 3;
}

int launch_stage(const Params& P, int n_batch, int stage, cudaStream_t s, cudaEvent_t* ev) {
  const unsigned nb = (unsigned)n_batch;
  // persistent chunk loops of T3 / T5: enough blocks to fill the machine across the batch
  const int per_event = max(8, 1184 / n_batch);
  LST_EV(0);
  switch (stage) {
    case LST_MD_: {
      dim3 g(min(per_event, P.L.n_chunk_hits), nb);
      k_md<false><<<g, kScanChunk, 0, s>>>(P);
      LST_EV(1);
      k_md<true><<<g, kScanChunk, 0, s>>>(P);
      break;
    }
    case LST_SEG_: {
      dim3 g(min(2 * per_event, P.L.n_chunk_md), nb);   // 128-thread blocks: twice as many per SM
      k_seg<<<g, kSegThreads, 0, s>>>(P);               // single pass (ticket + look-back)
      LST_EV(1);
      LST_EV(2);
      return 1;
    }
    case LST_T3_: {
      dim3 g(min(per_event, P.L.n_chunk_seg), nb);
      k_t3<false><<<g, kScanChunk, 0, s>>>(P);
      LST_EV(1);
      k_t3<true><<<g, kScanChunk, 0, s>>>(P);
      break;
    }
    case LST_T5_: {
      dim3 g(min(per_event, P.L.n_chunk_t3), nb);
      k_t5<false><<<g, kScanChunk, 0, s>>>(P);
      LST_EV(1);
      k_t5<true><<<g, kScanChunk, 0, s>>>(P);
      break;
    }
    default:
      return 0;
  }
  LST_EV(2);
  return 2;
}

int launch_gather_hits(const Params& P, int kind, int n, cudaStream_t s) {
  if (n <= 0) return 0;
  k_gather_hits<<<(n + 255) / 256, 256, 0, s>>>(P, kind, n);
  return 1;
}

int launch_pack_values(const Params& P, int kind, int n, cudaStream_t s) {
  if (n <= 0 || (kind != LST_MD_ && kind != LST_T3_)) return 0;
  k_pack_values<<<(n + 255) / 256, 256, 0, s>>>(P, kind, n);
  return 1;
}

}  // namespace lst
