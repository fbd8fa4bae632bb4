// ipa_prepare.cuh -- one-off data-layout preparation of the events: a STABLE counting sort on
// a coarse bin index,  bin(x) = clamp(floor((x - lo) IPA_PREP_BINS / (hi - lo)), 0, IPA_PREP_BINS - 1)  (NaN -> last bin).
//
// Why: the likelihood does not depend on the order of the events and the data of a fit are constant over the
// minimiser's calls.  The streaming kernels evaluate only the core polynomial or only the tail
// logarithm for a warp whose events all lie in one region, so events grouped by a fine enough bin index make
// nearly every warp region-uniform for EVERY theta of the fit (the bins do not depend on the joins).  The kernels
// only look at which side of a join an event lies on, so a full sort (8 radix passes over 64-bit keys) orders
// bits nobody reads; one counting pass on 11 bits does the same job.
//
// The result is a pure function of the input: the order inside a bin is the original order (stable), whatever the
// grid -- so the prepared array, and every NLL computed from it, is bitwise reproducible.  No floating-point
// arithmetic of the method happens here; the only integer atomics are histogram counts (order-independent).
//
//   ipa_prep_hist_kernel     block b counts the bins of its contiguous chunk            -> hist[bin][b]
//   ipa_prep_scan_kernel     per bin: exclusive prefix over the blocks, total per bin   -> hist (in place), bintot
//   ipa_prep_binscan_kernel  exclusive prefix over the bins                             -> binbase
//   ipa_prep_scatter_kernel  block b re-reads its chunk tile by tile, ranks every event inside its bin in original
//                            order (warp: match_any; block: per-warp counters + a scan over the warps) and writes
//                            it to  binbase[bin] + hist[bin][b] + rank
//   ipa_prep_segment_kernel  one block per segment (toy / category): the same three steps inside the segment
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define IPA_PREP_BINS 2048
#define IPA_PREP_THREADS 512
#define IPA_PREP_WARPS (IPA_PREP_THREADS / 32)
#define IPA_PREP_E 16                                   // events per thread and tile
#define IPA_PREP_TILE (IPA_PREP_THREADS * IPA_PREP_E)   // 8192 events: ranks inside a tile fit 16 bits
#define IPA_PREP_SMEM (IPA_PREP_WARPS * IPA_PREP_BINS * 2 + IPA_PREP_BINS * 8)

__device__ __forceinline__ int ipa_prep_bin(double x, double lo, double scale) {
  const double t = (x - lo) * scale;
  int b = (t < (double)IPA_PREP_BINS) ? (int)t : IPA_PREP_BINS - 1;     // NaN: the comparison is false -> last bin
  return b < 0 ? 0 : b;
}

// contiguous chunk of block b: whole tiles, so that every block but the last starts tile-aligned
__device__ __forceinline__ void ipa_prep_chunk(long long n, int b, int G, long long* beg, long long* end) {
  const long long tiles = (n + IPA_PREP_TILE - 1) / IPA_PREP_TILE;
  const long long per = (tiles + G - 1) / G;
  long long s = (long long)b * per * IPA_PREP_TILE, e = s + per * IPA_PREP_TILE;
  *beg = s < n ? s : n;
  *end = e < n ? e : n;
}

__global__ void __launch_bounds__(IPA_PREP_THREADS)
ipa_prep_hist_kernel(const double* __restrict__ x, long long n, double lo, double scale, unsigned int* __restrict__ hist) {
  __shared__ unsigned int cnt[IPA_PREP_BINS];
  for (int j = threadIdx.x; j < IPA_PREP_BINS; j += IPA_PREP_THREADS) cnt[j] = 0u;
  __syncthreads();
  long long beg, end;
  ipa_prep_chunk(n, blockIdx.x, gridDim.x, &beg, &end);
  long long i = beg + threadIdx.x;
  for (; i + 7LL * IPA_PREP_THREADS < end; i += 8LL * IPA_PREP_THREADS) {
    double v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) v[u] = __ldcs(x + i + (long long)u * IPA_PREP_THREADS);
#pragma unroll
    for (int u = 0; u < 8; ++u) atomicAdd(&cnt[ipa_prep_bin(v[u], lo, scale)], 1u);
  }
  for (; i < end; i += IPA_PREP_THREADS) atomicAdd(&cnt[ipa_prep_bin(__ldcs(x + i), lo, scale)], 1u);
  __syncthreads();
  for (int j = threadIdx.x; j < IPA_PREP_BINS; j += IPA_PREP_THREADS) hist[(long long)j * gridDim.x + blockIdx.x] = cnt[j];
}

// one warp per bin: exclusive prefix of hist[bin][0..G) in place, bintot[bin] = total
__global__ void __launch_bounds__(256)
ipa_prep_scan_kernel(unsigned int* __restrict__ hist, int G, unsigned long long* __restrict__ bintot) {
  const int lane = threadIdx.x & 31;
  const int bin = blockIdx.x * 8 + (threadIdx.x >> 5);
  if (bin >= IPA_PREP_BINS) return;
  unsigned int* row = hist + (long long)bin * G;
  unsigned long long run = 0;
  for (int base = 0; base < G; base += 32) {
    const int b = base + lane;
    const unsigned int c = b < G ? row[b] : 0u;
    unsigned int inc = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned int t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += t;
    }
    if (b < G) row[b] = (unsigned int)run + inc - c;        // a block's chunk holds < 2^32 events of one bin
    run += __shfl_sync(0xffffffffu, inc, 31);
  }
  if (lane == 0) bintot[bin] = run;
}

// one block: binbase[bin] = sum of bintot[0..bin)
__global__ void __launch_bounds__(IPA_PREP_THREADS)
ipa_prep_binscan_kernel(const unsigned long long* __restrict__ bintot, unsigned long long* __restrict__ binbase) {
  __shared__ unsigned long long part[IPA_PREP_THREADS];
  constexpr int PER = IPA_PREP_BINS / IPA_PREP_THREADS;
  unsigned long long v[PER], s = 0;
#pragma unroll
  for (int q = 0; q < PER; ++q) { v[q] = bintot[threadIdx.x * PER + q]; s += v[q]; }
  part[threadIdx.x] = s;
  __syncthreads();
  for (int o = 1; o < IPA_PREP_THREADS; o <<= 1) {
    const unsigned long long add = threadIdx.x >= o ? part[threadIdx.x - o] : 0ull;
    __syncthreads();
    part[threadIdx.x] += add;
    __syncthreads();
  }
  unsigned long long run = part[threadIdx.x] - s;
#pragma unroll
  for (int q = 0; q < PER; ++q) { binbase[threadIdx.x * PER + q] = run; run += v[q]; }
}

// Stable scatter of x[beg, end) given the running output position off[bin] (shared memory) of this block for every
// bin.  Tile by tile: (1) warp w ranks its 32 x E events -- event index inside the tile = (w E + e) 32 + lane, so
// (warp, e, lane) order IS the original order -- with match_any: rank inside the warp = events of the same bin seen
// before; the first lane of every match group bumps the warp's own 16-bit counter; (2) exclusive scan of the
// counters over the warps, two bins at a time (packed 16-bit pairs: a tile holds < 2^16 events); (3) every event
// goes to off[bin] + (events of the bin in earlier warps) + (rank in its warp); (4) off[bin] += tile count.
// wcnt [WARPS][BINS] uint16, off [BINS] uint64.
__device__ __forceinline__ void ipa_prep_scatter_range(const double* __restrict__ x, long long beg, long long end, double lo,
                                                       double scale, unsigned short* wcnt, unsigned long long* off,
                                                       double* __restrict__ out) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const unsigned lt = (1u << lane) - 1u;
  unsigned short* mine = wcnt + warp * IPA_PREP_BINS;
  unsigned int* wcnt32 = reinterpret_cast<unsigned int*>(wcnt);
  for (long long base = beg; base < end; base += IPA_PREP_TILE) {
    {  // zero the per-warp counters (128-bit stores)
      uint4* z = reinterpret_cast<uint4*>(wcnt);
      for (int i = tid; i < IPA_PREP_WARPS * IPA_PREP_BINS * 2 / 16; i += IPA_PREP_THREADS) z[i] = make_uint4(0u, 0u, 0u, 0u);
    }
    double v[IPA_PREP_E];
    const long long first = base + (long long)warp * (32 * IPA_PREP_E) + lane;
#pragma unroll
    for (int e = 0; e < IPA_PREP_E; ++e) {
      const long long i = first + 32 * e;
      v[e] = i < end ? __ldcs(x + i) : 0.0;
    }
    __syncthreads();
    unsigned short rank[IPA_PREP_E];
    short bin[IPA_PREP_E];
#pragma unroll
    for (int e = 0; e < IPA_PREP_E; ++e) {
      const bool live = first + 32 * e < end;
      const int b = live ? ipa_prep_bin(v[e], lo, scale) : -1;          // empty slots of the ragged tile match each other only
      const unsigned peers = __match_any_sync(0xffffffffu, b);
      const int leader = __ffs(peers) - 1;
      unsigned old = 0;
      if (lane == leader && live) {
        old = mine[b];
        mine[b] = (unsigned short)(old + __popc(peers));
      }
      old = __shfl_sync(0xffffffffu, old, leader);
      rank[e] = (unsigned short)(old + __popc(peers & lt));
      bin[e] = (short)b;
      __syncwarp();
    }
    __syncthreads();
    // exclusive scan over the warps, bins (2 q, 2 q + 1) packed in one 32-bit word; thread owns words q = tid + i 512
    unsigned int tot[IPA_PREP_BINS / 2 / IPA_PREP_THREADS];
#pragma unroll
    for (int i = 0; i < IPA_PREP_BINS / 2 / IPA_PREP_THREADS; ++i) {
      const int q = tid + i * IPA_PREP_THREADS;
      unsigned int run = 0;
#pragma unroll
      for (int w = 0; w < IPA_PREP_WARPS; ++w) {
        const unsigned int c = wcnt32[w * (IPA_PREP_BINS / 2) + q];
        wcnt32[w * (IPA_PREP_BINS / 2) + q] = run;
        run += c;                                                         // no carry between the halves: sums < 2^16
      }
      tot[i] = run;
    }
    __syncthreads();
#pragma unroll
    for (int e = 0; e < IPA_PREP_E; ++e) {
      if (bin[e] >= 0) out[off[bin[e]] + mine[bin[e]] + rank[e]] = v[e];
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < IPA_PREP_BINS / 2 / IPA_PREP_THREADS; ++i) {
      const int q = tid + i * IPA_PREP_THREADS;
      off[2 * q] += tot[i] & 0xffffu;
      off[2 * q + 1] += tot[i] >> 16;
    }
    // no barrier here: the next tile zeroes wcnt (free since the barrier above) and reads off[] two barriers later
  }
}

__global__ void __launch_bounds__(IPA_PREP_THREADS)
ipa_prep_scatter_kernel(const double* __restrict__ x, long long n, double lo, double scale,
                        const unsigned int* __restrict__ hist, const unsigned long long* __restrict__ binbase,
                        double* __restrict__ out) {
  extern __shared__ __align__(16) unsigned char ipa_prep_smem[];
  unsigned short* wcnt = reinterpret_cast<unsigned short*>(ipa_prep_smem);
  unsigned long long* off = reinterpret_cast<unsigned long long*>(ipa_prep_smem + IPA_PREP_WARPS * IPA_PREP_BINS * 2);
  for (int j = threadIdx.x; j < IPA_PREP_BINS; j += IPA_PREP_THREADS)
    off[j] = binbase[j] + hist[(long long)j * gridDim.x + blockIdx.x];
  __syncthreads();
  long long beg, end;
  ipa_prep_chunk(n, blockIdx.x, gridDim.x, &beg, &end);
  ipa_prep_scatter_range(x, beg, end, lo, scale, wcnt, off, out);
}

// One block per segment: histogram of the segment, exclusive prefix over the bins, stable scatter inside the segment.
__global__ void __launch_bounds__(IPA_PREP_THREADS)
ipa_prep_segment_kernel(const double* __restrict__ x, const long long* __restrict__ offsets, double lo, double scale,
                        double* __restrict__ out) {
  extern __shared__ __align__(16) unsigned char ipa_prep_smem[];
  unsigned short* wcnt = reinterpret_cast<unsigned short*>(ipa_prep_smem);
  unsigned long long* off = reinterpret_cast<unsigned long long*>(ipa_prep_smem + IPA_PREP_WARPS * IPA_PREP_BINS * 2);
  unsigned int* cnt = reinterpret_cast<unsigned int*>(ipa_prep_smem);          // the counters' area, before it is needed
  __shared__ unsigned long long part[IPA_PREP_THREADS];
  const long long beg = offsets[blockIdx.x], end = offsets[blockIdx.x + 1];
  for (int j = threadIdx.x; j < IPA_PREP_BINS; j += IPA_PREP_THREADS) cnt[j] = 0u;
  __syncthreads();
  for (long long i = beg + threadIdx.x; i < end; i += IPA_PREP_THREADS) atomicAdd(&cnt[ipa_prep_bin(x[i], lo, scale)], 1u);
  __syncthreads();
  constexpr int PER = IPA_PREP_BINS / IPA_PREP_THREADS;
  unsigned long long v[PER], s = 0;
#pragma unroll
  for (int q = 0; q < PER; ++q) { v[q] = cnt[threadIdx.x * PER + q]; s += v[q]; }
  part[threadIdx.x] = s;
  __syncthreads();
  for (int o = 1; o < IPA_PREP_THREADS; o <<= 1) {
    const unsigned long long add = threadIdx.x >= o ? part[threadIdx.x - o] : 0ull;
    __syncthreads();
    part[threadIdx.x] += add;
    __syncthreads();
  }
  unsigned long long run = (unsigned long long)beg + part[threadIdx.x] - s;
#pragma unroll
  for (int q = 0; q < PER; ++q) { off[threadIdx.x * PER + q] = run; run += v[q]; }
  __syncthreads();
  ipa_prep_scatter_range(x, beg, end, lo, scale, wcnt, off, out);
}
