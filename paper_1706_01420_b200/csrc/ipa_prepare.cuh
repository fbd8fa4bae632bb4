// ipa_prepare.cuh -- one-off data-layout preparation of the events: a STABLE counting sort on
// a coarse bin index,  bin(x) = clamp(floor((x - lo) IPA_PREP_BINS / (hi - lo)), 0, IPA_PREP_BINS - 1)  (NaN -> last bin).
//
// Why: the likelihood does not depend on the order of the events and the data of a fit are constant over the
// minimiser's calls.  The streaming kernels evaluate only the core polynomial or only the tail
// logarithm for a warp whose events all lie in one region, so events grouped by a fine enough bin index make
// nearly every warp region-uniform for EVERY theta of the fit (the bins do not depend on the joins).  The kernels
// only look at which side of a join an event lies on, so a full sort (8 radix passes over 64-bit keys) orders
// bits nobody reads; ONE counting pass on 8 bits does the same job: only the warps inside the two bins that hold a
// join stay mixed (2 / 256 of the range: about 1 % of the events of the config model).
//
// The result is a pure function of the input: the order inside a bin is the original order (stable), whatever the
// grid -- so the prepared array, and every NLL computed from it, is bitwise reproducible.  No floating-point
// arithmetic of the method happens here; the only integer atomics are histogram counts (order-independent).
//
//   ipa_prep_hist_kernel     block b counts the bins of its contiguous chunk            -> hist[bin][b]
//   ipa_prep_scan_kernel     per bin: exclusive prefix over the blocks, total per bin   -> hist (in place), bintot
//   ipa_prep_binscan_kernel  exclusive prefix over the bins                             -> binbase
//   ipa_prep_scatter_kernel  block b re-reads its chunk tile by tile (4096 events): ranks every event inside its bin
//                            in original order (warp: ballots on the bits of the bin; block: per-warp counters + a scan over the warps),
//                            moves the tile into bin order in SHARED memory and writes it out in runs of consecutive
//                            addresses (one run per bin), starting at  binbase[bin] + hist[bin][b]
//   ipa_prep_segment_kernel  one block per segment (toy / category): the same three steps inside the segment
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define IPA_PREP_BINS 256                               // == IPA_PREPARE_BINS of the header (asserted in ipa_api.cu)
#define IPA_PREP_THREADS 512                           // measured per 1e8 events: 256 x 6 blocks per SM 0.88 ms, 256 x 4 0.83, 512 x 2 0.79, 512 x 3 0.78, 1024 x 1 0.81
#define IPA_PREP_BLOCKS_PER_SM 3                       // 40 registers, 62 KB of shared memory per block
#define IPA_PREP_WARPS (IPA_PREP_THREADS / 32)
#define IPA_PREP_E 8                                    // events per thread and tile
#define IPA_PREP_TILE (IPA_PREP_THREADS * IPA_PREP_E)   // 4096 events: ranks and positions inside a tile fit 16 bits
// dynamic shared memory of the scatter: stage [TILE] double | off [BINS] u64 | delta [BINS] u64 | tilebase [BINS] u32 |
// wtot [8] u32 | wmap [WARPS][BINS] u32 | wcnt [WARPS][BINS] u16 | sbin [TILE] u8
#define IPA_PREP_SMEM (IPA_PREP_TILE * 8 + IPA_PREP_BINS * 16 + (IPA_PREP_BINS + 8) * 4 + IPA_PREP_WARPS * IPA_PREP_BINS * 6 + \
                       IPA_PREP_TILE + 64)
static_assert(IPA_PREP_BINS == 256 && IPA_PREP_THREADS >= IPA_PREP_BINS, "one thread per bin in the block scans");

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
  // per-WARP private counters (a block-wide array of 256 counters serialises on the few bins under the peak)
  __shared__ unsigned int cnt[IPA_PREP_WARPS][IPA_PREP_BINS];
  unsigned int* mine = cnt[threadIdx.x >> 5];
  for (int j = threadIdx.x; j < IPA_PREP_WARPS * IPA_PREP_BINS; j += IPA_PREP_THREADS) (&cnt[0][0])[j] = 0u;
  __syncthreads();
  long long beg, end;
  ipa_prep_chunk(n, blockIdx.x, gridDim.x, &beg, &end);
  long long i = beg + threadIdx.x;
  for (; i + 7LL * IPA_PREP_THREADS < end; i += 8LL * IPA_PREP_THREADS) {
    double v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) v[u] = __ldcs(x + i + (long long)u * IPA_PREP_THREADS);
#pragma unroll
    for (int u = 0; u < 8; ++u) atomicAdd(&mine[ipa_prep_bin(v[u], lo, scale)], 1u);
  }
  for (; i < end; i += IPA_PREP_THREADS) atomicAdd(&mine[ipa_prep_bin(__ldcs(x + i), lo, scale)], 1u);
  __syncthreads();
  for (int j = threadIdx.x; j < IPA_PREP_BINS; j += IPA_PREP_THREADS) {
    unsigned int s = 0;
#pragma unroll
    for (int w = 0; w < IPA_PREP_WARPS; ++w) s += cnt[w][j];
    hist[(long long)j * gridDim.x + blockIdx.x] = s;
  }
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
    if (b < G) row[b] = (unsigned int)run + inc - c;        // a bin holds < 2^32 events (n <= 2^32 - 1)
    run += __shfl_sync(0xffffffffu, inc, 31);
  }
  if (lane == 0) bintot[bin] = run;
}

// one block of IPA_PREP_BINS threads: binbase[bin] = sum of bintot[0..bin)
__global__ void __launch_bounds__(IPA_PREP_BINS)
ipa_prep_binscan_kernel(const unsigned long long* __restrict__ bintot, unsigned long long* __restrict__ binbase) {
  __shared__ unsigned long long part[IPA_PREP_BINS];
  const unsigned long long v = bintot[threadIdx.x];
  part[threadIdx.x] = v;
  __syncthreads();
  for (int o = 1; o < IPA_PREP_BINS; o <<= 1) {
    const unsigned long long add = threadIdx.x >= o ? part[threadIdx.x - o] : 0ull;
    __syncthreads();
    part[threadIdx.x] += add;
    __syncthreads();
  }
  binbase[threadIdx.x] = part[threadIdx.x] - v;
}

struct IpaPrepSmem {
  double* stage;                 // [TILE]  the tile in bin order
  unsigned long long* off;       // [BINS]  running output position of this block for every bin
  unsigned long long* delta;     // [BINS]  off - tilebase: output address of a staged position = delta[bin] + position
  unsigned int* wmap;            // [WARPS][BINS] lanes of the warp that hold the bin in the current step (bit mask)
  unsigned int* tilebase;        // [BINS]  first staged position of a bin in the current tile
  unsigned short* wcnt;          // [WARPS][BINS] events of a bin per warp, then their exclusive prefix over the warps
  unsigned char* sbin;           // [TILE]  bin of the staged event
  unsigned int* wtot;            // [8]     warp totals of the scan over the bins
};
__device__ __forceinline__ IpaPrepSmem ipa_prep_carve(unsigned char* base) {
  IpaPrepSmem m;
  m.stage = reinterpret_cast<double*>(base);
  unsigned char* p = base + IPA_PREP_TILE * 8;
  m.off = reinterpret_cast<unsigned long long*>(p);      p += IPA_PREP_BINS * 8;
  m.delta = reinterpret_cast<unsigned long long*>(p);    p += IPA_PREP_BINS * 8;
  m.tilebase = reinterpret_cast<unsigned int*>(p);       p += IPA_PREP_BINS * 4;
  m.wtot = reinterpret_cast<unsigned int*>(p);           p += 32;
  m.wmap = reinterpret_cast<unsigned int*>(p);           p += IPA_PREP_WARPS * IPA_PREP_BINS * 4;
  m.wcnt = reinterpret_cast<unsigned short*>(p);         p += IPA_PREP_WARPS * IPA_PREP_BINS * 2;
  m.sbin = p;
  return m;
}

// Stable scatter of x[beg, end) given the running output position off[bin] (shared memory) of this block for every
// bin.  Tile by tile: (1) warp w ranks its 32 x E events -- event index inside the tile = (w E + e) 32 + lane, so
// (warp, e, lane) order IS the original order -- by ballots: rank inside the warp = events of the same bin seen
// before; the first lane of every match group bumps the warp's own 16-bit counter; (2) thread b: exclusive prefix of
// bin b's counters over the warps, then an exclusive scan of the tile's bin counts over the bins; (3) every event
// goes to stage[tilebase[bin] + (events of the bin in earlier warps) + (rank in its warp)]: the tile in bin order,
// original order inside a bin; (4) the staged tile is written out position by position: consecutive positions of a
// bin are consecutive addresses, off[bin] + (position - tilebase[bin]); (5) off[bin] += tile count.
__device__ __forceinline__ void ipa_prep_scatter_range(const double* __restrict__ x, long long beg, long long end, double lo,
                                                       double scale, const IpaPrepSmem& m, double* __restrict__ out) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const unsigned lt = (1u << lane) - 1u;
  unsigned short* mine = m.wcnt + warp * IPA_PREP_BINS;
  unsigned int* map = m.wmap + warp * IPA_PREP_BINS;
  for (int i = tid; i < IPA_PREP_WARPS * IPA_PREP_BINS; i += IPA_PREP_THREADS) m.wmap[i] = 0u;   // kept zero by the leaders
  const int first = warp * (32 * IPA_PREP_E) + lane;
  // the events of a tile are loaded one tile ahead (right after the previous tile has been staged, when v[] is free): the
  // loads fly during the write-out of the previous tile and the zeroing below
  double v[IPA_PREP_E], vn[IPA_PREP_E];
#pragma unroll
  for (int e = 0; e < IPA_PREP_E; ++e) vn[e] = (beg + first + 32 * e < end) ? __ldcs(x + beg + first + 32 * e) : 0.0;
  for (long long base = beg; base < end; base += IPA_PREP_TILE) {
    const int cnt = (int)((end - base < IPA_PREP_TILE) ? (end - base) : IPA_PREP_TILE);
    {  // zero the per-warp counters (128-bit stores)
      uint4* z = reinterpret_cast<uint4*>(m.wcnt);
      for (int i = tid; i < IPA_PREP_WARPS * IPA_PREP_BINS * 2 / 16; i += IPA_PREP_THREADS) z[i] = make_uint4(0u, 0u, 0u, 0u);
    }
#pragma unroll
    for (int e = 0; e < IPA_PREP_E; ++e) v[e] = vn[e];
    __syncthreads();
    unsigned int key[IPA_PREP_E];               // bin << 16 | rank inside the warp
    const bool full = cnt == IPA_PREP_TILE;
#pragma unroll
    for (int e = 0; e < IPA_PREP_E; ++e) {
      const bool live = full || first + 32 * e < cnt;
      const unsigned b = live ? (unsigned)ipa_prep_bin(v[e], lo, scale) : 0u;
      // lanes of the warp holding the same bin, through the warp's own bit map in shared memory: every live lane ORs
      // its bit into map[bin] (an OR does not depend on the order the hardware takes the lanes in: deterministic),
      // reads the mask back, and the first lane of the mask bumps the warp's counter of the bin and clears the map
      // entry.  3 shared-memory instructions where eight ballots and their logic took 50, and the match.any
      // instruction serialised on the ~25 distinct bins of a warp of unsorted events.
      if (live) atomicOr(&map[b], 1u << lane);
      __syncwarp();
      const unsigned peers = live ? map[b] : 0u;
      __syncwarp();
      const int leader = __ffs(peers) - 1;
      unsigned old = 0;
      if (live && lane == leader) {
        old = mine[b];
        mine[b] = (unsigned short)(old + __popc(peers));
        map[b] = 0u;
      }
      old = __shfl_sync(0xffffffffu, old, leader & 31);
      key[e] = (b << 16) | (old + __popc(peers & lt));
      __syncwarp();
    }
    __syncthreads();
    // thread b: exclusive prefix of bin b over the warps; then exclusive scan of the tile counts over the bins
    unsigned int tot = 0;
    if (tid < IPA_PREP_BINS) {
#pragma unroll
      for (int w = 0; w < IPA_PREP_WARPS; ++w) {
        const unsigned int c = m.wcnt[w * IPA_PREP_BINS + tid];
        m.wcnt[w * IPA_PREP_BINS + tid] = (unsigned short)tot;
        tot += c;
      }
      unsigned int inc = tot;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
      }
      if (lane == 31) m.wtot[warp] = inc;
      m.tilebase[tid] = inc - tot;                       // exclusive inside the warp; the warp offset is added below
    }
    __syncthreads();
    if (tid < IPA_PREP_BINS) {
      unsigned int add = 0;
      for (int w = 0; w < warp; ++w) add += m.wtot[w];
      const unsigned int tb = m.tilebase[tid] + add;
      m.tilebase[tid] = tb;
      m.delta[tid] = m.off[tid] - tb;
    }
    __syncthreads();
#pragma unroll
    for (int e = 0; e < IPA_PREP_E; ++e) {
      if (full || first + 32 * e < cnt) {
        const unsigned int b = key[e] >> 16;
        const unsigned int pos = m.tilebase[b] + mine[b] + (key[e] & 0xffffu);
        m.stage[pos] = v[e];
        m.sbin[pos] = (unsigned char)b;
      }
    }
    {
      const long long nb = base + IPA_PREP_TILE;
#pragma unroll
      for (int e = 0; e < IPA_PREP_E; ++e) vn[e] = (nb + first + 32 * e < end) ? __ldcs(x + nb + first + 32 * e) : 0.0;
    }
    __syncthreads();
    for (int i = tid; i < cnt; i += IPA_PREP_THREADS) {
      out[m.delta[m.sbin[i]] + (unsigned int)i] = m.stage[i];
    }
    __syncthreads();
    if (tid < IPA_PREP_BINS) m.off[tid] += tot;
    // no barrier here: the next tile touches wcnt (free since the staging barrier) and reads off[] three barriers later
  }
}

__global__ void __launch_bounds__(IPA_PREP_THREADS, IPA_PREP_BLOCKS_PER_SM)
ipa_prep_scatter_kernel(const double* __restrict__ x, long long n, double lo, double scale,
                        const unsigned int* __restrict__ hist, const unsigned long long* __restrict__ binbase,
                        double* __restrict__ out) {
  extern __shared__ __align__(16) unsigned char ipa_prep_smem[];
  const IpaPrepSmem m = ipa_prep_carve(ipa_prep_smem);
  if (threadIdx.x < IPA_PREP_BINS) m.off[threadIdx.x] = binbase[threadIdx.x] + hist[(long long)threadIdx.x * gridDim.x + blockIdx.x];
  __syncthreads();
  long long beg, end;
  ipa_prep_chunk(n, blockIdx.x, gridDim.x, &beg, &end);
  ipa_prep_scatter_range(x, beg, end, lo, scale, m, out);
}

// One block per segment: histogram of the segment, exclusive prefix over the bins, stable scatter inside the segment.
__global__ void __launch_bounds__(IPA_PREP_THREADS, IPA_PREP_BLOCKS_PER_SM)
ipa_prep_segment_kernel(const double* __restrict__ x, const long long* __restrict__ offsets, double lo, double scale,
                        double* __restrict__ out) {
  extern __shared__ __align__(16) unsigned char ipa_prep_smem[];
  const IpaPrepSmem m = ipa_prep_carve(ipa_prep_smem);
  unsigned int* cnt = reinterpret_cast<unsigned int*>(m.stage);              // [WARPS][BINS] in the staging area, before it is needed
  __shared__ unsigned long long part[IPA_PREP_BINS];
  const int tid = threadIdx.x;
  const long long beg = offsets[blockIdx.x], end = offsets[blockIdx.x + 1];
  for (int j = tid; j < IPA_PREP_WARPS * IPA_PREP_BINS; j += IPA_PREP_THREADS) cnt[j] = 0u;
  __syncthreads();
  unsigned int* mine = cnt + (tid >> 5) * IPA_PREP_BINS;
  for (long long i = beg + tid; i < end; i += IPA_PREP_THREADS) atomicAdd(&mine[ipa_prep_bin(x[i], lo, scale)], 1u);
  __syncthreads();
  unsigned long long v = 0;
  if (tid < IPA_PREP_BINS) {
    for (int w = 0; w < IPA_PREP_WARPS; ++w) v += cnt[w * IPA_PREP_BINS + tid];
    part[tid] = v;
  }
  __syncthreads();
  for (int o = 1; o < IPA_PREP_BINS; o <<= 1) {
    unsigned long long add = 0ull;
    if (tid < IPA_PREP_BINS && tid >= o) add = part[tid - o];
    __syncthreads();
    if (tid < IPA_PREP_BINS) part[tid] += add;
    __syncthreads();
  }
  if (tid < IPA_PREP_BINS) m.off[tid] = (unsigned long long)beg + part[tid] - v;
  __syncthreads();
  ipa_prep_scatter_range(x, beg, end, lo, scale, m, out);
}
