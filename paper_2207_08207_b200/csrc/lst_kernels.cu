// lst_kernels.cu -- sm_100a kernels of the LST hot path (DESIGN.md sections 5-6).
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
// a0: load + bin by (module, side) + order by original index + derive r
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_bin_count(const __grid_constant__ Params P, const HitInput in) {
  Slot S(P, 0);
  unsigned* cnt = S.bin_start();
  int bad = 0;
  for (int h = blockIdx.x * blockDim.x + threadIdx.x; h < in.n; h += gridDim.x * blockDim.x) {
    const int m = in.module[h];
    const unsigned sd = in.side[h];
    if (m < 0 || m >= P.L.n_modules || sd > 1u) { ++bad; continue; }
    atomicAdd(cnt + (2 * m + (int)sd), 1u);
  }
  if (bad) atomicAdd(&S.hdr()->bad_hits, bad);
}

__global__ void __launch_bounds__(1024) k_bin_scan(const __grid_constant__ Params P) {
  Slot S(P, 0);
  int* start = reinterpret_cast<int*>(S.bin_start());
  const int total = block_scan_array<1024>(start, P.L.n_bins, -1);
  __syncthreads();
  // candidate count of the MD stage: sum over modules of (#lower hits) x (#upper hits)
  unsigned long long c = 0;
  for (int m = threadIdx.x; m < P.L.n_modules; m += 1024) {
    const unsigned long long l = start[2 * m + 1] - start[2 * m], u = start[2 * m + 2] - start[2 * m + 1];
    c += l * u;
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) c += __shfl_down_sync(0xffffffffu, c, d);
  if (lane_id() == 0 && c) atomicAdd(&S.hdr()->cand[LST_MD_], c);
  if (threadIdx.x == 0) S.hdr()->n_hits = total;
}

__global__ void __launch_bounds__(256) k_bin_scatter(const __grid_constant__ Params P, const HitInput in) {
  Slot S(P, 0);
  const unsigned* start = S.bin_start();
  unsigned* cur = S.bin_cursor();
  int* tmp = S.tmp_idx();
  for (int h = blockIdx.x * blockDim.x + threadIdx.x; h < in.n; h += gridDim.x * blockDim.x) {
    const int m = in.module[h];
    const unsigned sd = in.side[h];
    if (m < 0 || m >= P.L.n_modules || sd > 1u) continue;
    const int b = 2 * m + (int)sd;
    tmp[start[b] + atomicAdd(cur + b, 1u)] = h;
  }
}

// One warp per bin: rank the bin's original indices (ascending) and gather the coordinates.
__global__ void __launch_bounds__(256) k_bin_order(const __grid_constant__ Params P, const HitInput in) {
  Slot S(P, 0);
  const int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (b >= P.L.n_bins) return;
  const unsigned* start = S.bin_start();
  const int s = start[b], n = start[b + 1] - s;
  const int* tmp = S.tmp_idx() + s;
  float4* hit4 = S.hit4() + s;
  int* orig = S.hit_orig() + s;
  for (int i = lane_id(); i < n; i += 32) {
    const int mine = tmp[i];
    int rank = 0;
    for (int j = 0; j < n; ++j) rank += (tmp[j] < mine);
    const float x = in.x[mine], y = in.y[mine], z = in.z[mine];
    hit4[rank] = make_float4(x, y, z, sqrtf(x * x + y * y));
    orig[rank] = mine;
  }
}

// ------------------------------------------------------------------------------------------
// a1: mini-doublets. One warp per module; lanes sweep the (lower, upper) pairs of the module
// in row-major order p = l * U + u.
// ------------------------------------------------------------------------------------------
constexpr int kMdWarps = 8;

template <bool FILL>
__global__ void __launch_bounds__(kMdWarps * 32) k_md(const __grid_constant__ Params P) {
  Slot S(P, blockIdx.y);
  const int m = blockIdx.x * kMdWarps + (threadIdx.x >> 5);
  int* md_start = S.md_start();
  if (m < P.L.n_modules) {
    const unsigned* bs = S.bin_start();
    const unsigned s0 = bs[2 * m], s1 = bs[2 * m + 1], s2 = bs[2 * m + 2];
    const unsigned L = s1 - s0, U = s2 - s1, T = L * U;
    const int layer = P.mod_layer[m];
    const float4* hit4 = S.hit4();
    int running = 0;
    const int base = FILL ? md_start[m] : 0;
    for (unsigned p0 = 0; p0 < T; p0 += 32) {
      const unsigned p = p0 + lane_id();
      bool pass = false;
      float4 lo, up;
      MdOut o;
      unsigned l = 0, u = 0;
      if (p < T) {
        l = p / U;
        u = p - l * U;
        lo = hit4[s0 + l];
        up = hit4[s1 + u];
        pass = md_select(P.cuts, layer, lo, up, o);
      }
      const unsigned bal = __ballot_sync(0xffffffffu, pass);
      if (FILL && pass) {
        const int pos = base + running + __popc(bal & lanemask_lt());
        if (pos < P.L.cap_md) {
          S.md_anchor()[pos] = lo;
          S.md_aux()[pos] = make_float2(up.w, o.sinA);
          S.md_hits()[pos] = make_int2(S.hit_orig()[s0 + l], S.hit_orig()[s1 + u]);
          S.md_out()[pos] = make_float2(atan2f(lo.x * up.y - lo.y * up.x, lo.x * up.x + lo.y * up.y),
                                        atan2f(o.cross, o.dot));
          S.md_module()[pos] = m;
        }
      }
      running += __popc(bal);
    }
    if (!FILL && lane_id() == 0) md_start[m] = running;
  }
  if (!FILL) {
    if (last_block_done(&S.hdr()->done[0], gridDim.x)) {
      const int total = block_scan_array<kMdWarps * 32>(md_start, P.L.n_modules, P.L.cap_md);
      if (threadIdx.x == 0) publish_total(S.hdr(), LST_MD_, total, P.L.cap_md);
    }
  }
}

// ------------------------------------------------------------------------------------------
// a2: segments. One block per inner module A; one warp per inner MD at a time; lanes sweep the
// outer MDs of the modules connected to A.  The module map is stored as runs of consecutive
// target modules, and MDs are stored in module order, so every run is ONE contiguous range of
// MD indices: coalesced 16-B loads, no per-module indirection.
// ------------------------------------------------------------------------------------------
constexpr int kSegThreads = 128;

template <bool FILL>
__global__ void __launch_bounds__(kSegThreads) k_seg(const __grid_constant__ Params P) {
  Slot S(P, blockIdx.y);
  const int A = blockIdx.x;
  const int* md_start = S.md_start();
  int* seg_start = S.seg_start();
  const int mdLo = md_start[A], nA = md_start[A + 1] - mdLo;
  const int r0 = P.run_offsets[A], r1 = P.run_offsets[A + 1];
  const int layer = P.mod_layer[A];
  const float4* anchor = S.md_anchor();
  const float2* aux = S.md_aux();
  const int warp = threadIdx.x >> 5;
  const int blockBase = FILL ? S.seg_block_base()[A] : 0;
  unsigned long long nOut = 0;
  for (int k = warp; k < nA; k += kSegThreads / 32) {
    const int i = mdLo + k;
    const float4 ai = anchor[i];
    const float2 xi = aux[i];
    int running = 0;
    const int base = FILL ? blockBase + seg_start[i] : 0;
    for (int r = r0; r < r1; ++r) {
      const int2 run = P.runs[r];
      const int lo = md_start[run.x], hi = md_start[run.y + 1];
      if (k == warp) nOut += (unsigned long long)(hi - lo);
      for (int o0 = lo; o0 < hi; o0 += 32) {
        const int o = o0 + lane_id();
        bool pass = false;
        SegOut so;
        float4 ao;
        if (o < hi) {
          ao = anchor[o];
          const float2 xo = aux[o];
          pass = seg_select(P.cuts, layer, ai, xi, ao, xo, so);
        }
        const unsigned bal = __ballot_sync(0xffffffffu, pass);
        if (FILL && pass) {
          const int pos = base + running + __popc(bal & lanemask_lt());
          if (pos < P.L.cap_seg) {
            S.seg_md()[pos] = make_int2(i, o);
            S.seg_f()[pos] = make_float4(so.sinS, so.z0,
                                         atan2f(ai.x * ao.y - ai.y * ao.x, ai.x * ao.x + ai.y * ao.y),
                                         atan2f(so.cross, so.dot));
          }
        }
        running += __popc(bal);
      }
    }
    __syncwarp();  // every lane has read seg_start[i] (the local offset) before it is replaced
    if (lane_id() == 0) seg_start[i] = FILL ? min(base, P.L.cap_seg) : running;
  }
  if (FILL) return;
  // block-local exclusive scan of the per-MD counts (in place), block total -> seg_block_base[A]
  __syncthreads();
  int carry = 0;
  for (int k0 = 0; k0 < nA; k0 += kSegThreads) {
    const int k = k0 + threadIdx.x;
    const int v = (k < nA) ? seg_start[mdLo + k] : 0;
    int tot;
    const int ex = block_excl_scan<kSegThreads>(v, tot);
    if (k < nA) seg_start[mdLo + k] = carry + ex;
    carry += tot;
  }
  if (threadIdx.x == 0) {
    S.seg_block_base()[A] = carry;
    if (nA > 0 && nOut) atomicAdd(&S.hdr()->cand[LST_SEG_], nOut * (unsigned long long)nA);
  }
  if (last_block_done(&S.hdr()->done[1], gridDim.x)) {
    const int total = block_scan_array<kSegThreads>(S.seg_block_base(), P.L.n_modules, -1);
    if (threadIdx.x == 0) {
      publish_total(S.hdr(), LST_SEG_, total, P.L.cap_seg);
      seg_start[S.hdr()->n[LST_MD_]] = min(total, P.L.cap_seg);
    }
  }
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
    if (lane_id() == 0 && cand) atomicAdd(&H->cand[LST_T3_], cand);
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
    if (lane_id() == 0 && cand) atomicAdd(&H->cand[LST_T5_], cand);
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

int launch_bin(const Params& P, const HitInput& in, cudaStream_t s, cudaEvent_t* ev) {
  const int nb = in.n > 0 ? min((in.n + 255) / 256, 1184) : 0;
  int launches = 0;
  LST_EV(0);
  if (nb) { k_bin_count<<<nb, 256, 0, s>>>(P, in); ++launches; }
  LST_EV(1);
  k_bin_scan<<<1, 1024, 0, s>>>(P); ++launches;
  LST_EV(2);
  if (nb) { k_bin_scatter<<<nb, 256, 0, s>>>(P, in); ++launches; }
  LST_EV(3);
  if (nb) { k_bin_order<<<(P.L.n_bins + 7) / 8, 256, 0, s>>>(P, in); ++launches; }
  LST_EV(4);
  return launches;
}

int launch_stage(const Params& P, int n_batch, int stage, cudaStream_t s, cudaEvent_t* ev) {
  const unsigned nb = (unsigned)n_batch;
  // persistent chunk loops of T3 / T5: enough blocks to fill the machine across the batch
  const int per_event = max(8, 1184 / n_batch);
  LST_EV(0);
  switch (stage) {
    case LST_MD_: {
      dim3 g((P.L.n_modules + kMdWarps - 1) / kMdWarps, nb);
      k_md<false><<<g, kMdWarps * 32, 0, s>>>(P);
      LST_EV(1);
      k_md<true><<<g, kMdWarps * 32, 0, s>>>(P);
      break;
    }
    case LST_SEG_: {
      dim3 g(P.L.n_modules, nb);
      k_seg<false><<<g, kSegThreads, 0, s>>>(P);
      LST_EV(1);
      k_seg<true><<<g, kSegThreads, 0, s>>>(P);
      break;
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
