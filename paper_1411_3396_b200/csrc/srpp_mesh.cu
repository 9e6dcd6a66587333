// srpp_mesh.cu -- chaining-mesh binning (steps A1-A4 of SURVEY.md 8(a)) for sm_100a.
//
// The mesh is a STABLE counting sort of the particles by linear cell id (readings R10-R12):
//   A1  cell id per particle, fp32:  c = min((int)floorf(x * inv), ncell-1), inv = (float)ncell/box
//   A2-A4 histogram / exclusive scan / stable scatter.  A cell id has up to 24 bits and single cells hold
//        millions of particles, so the counting sort is applied digit-wise, least significant digit first,
//        in digits of <= 8 bits (three passes cover the 2^24-cell limit) and with the particle PAYLOAD
//        (float4 position+mass and original index) carried through every pass.  All global traffic is
//        streaming: each pass reads its input once, coalesced, re-orders a 4096-element tile by digit in
//        shared memory, and writes per-digit runs.  No random gather remains (the first version sorted
//        (key, index) pairs and gathered float4 through perm at the end: 32-byte sectors for 16 useful bytes).
//        Ranks inside a tile come from warp match + per-warp digit counters in warp-major order, so no atomic
//        decides an output position: perm is bit-exact reproducible and equals the oracle's stable
//        counting sort.
//   cell_start = run boundaries of the sorted ids (= exclusive prefix sum of the cell histogram).
// Per pass: [per-tile digit histogram (fused into A1 for the first pass)] -> column scan over tiles ->
// scatter.  Algorithmic bytes per build: 52*N + 8*ncells; moved by this design for three
// passes: 20 + 44 + 4 + 48 + 4 + 48 + 4 = 172 bytes per particle, all coalesced.  (Two passes of 10-bit digits move
// 120 bytes, but a 4096-element tile then writes 4-element runs per digit: the partially covered 32-byte sectors cost
// more DRAM read-modify-write traffic than the third pass -- measured.)
// Paper context: PAPER.md:63/65 (direct PP short-range solver inside the hand-over radius); the chaining
// mesh itself is named by BASELINE.json north_star.
#include <algorithm>

#include "srpp_internal.cuh"

namespace srpp {

// ------------------------------------------------------------------------------ small block helpers --
// Exclusive scan of one value per thread over a kSortThreads-wide CTA; `scratch` holds kSortWarps words.
__device__ __forceinline__ uint32_t cta_exclusive_scan(uint32_t v, uint32_t* scratch) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
    if (lane >= o) x += y;
  }
  __syncthreads();                       // scratch may still be read by a previous call
  if (lane == 31) scratch[wid] = x;
  __syncthreads();
  if (wid == 0) {
    uint32_t w = lane < kSortWarps ? scratch[lane] : 0u;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t y = __shfl_up_sync(0xffffffffu, w, o);
      if (lane >= o) w += y;
    }
    if (lane < kSortWarps) scratch[lane] = w;   // inclusive over warps
  }
  __syncthreads();
  return (wid ? scratch[wid - 1] : 0u) + (x - v);
}

// In-place exclusive scan of a[0..nbins) in shared memory (nbins a power of two, 32 <= nbins <= kSortMaxBins).
__device__ __forceinline__ void cta_scan_bins(uint32_t* a, int nbins, uint32_t* scratch) {
  const int per = nbins > kSortThreads ? nbins / kSortThreads : 1;   // 1, 2 or 4
  const int b0 = threadIdx.x * per;
  uint32_t v[kSortBinsPerThread], s = 0;
#pragma unroll
  for (int j = 0; j < kSortBinsPerThread; ++j) {
    v[j] = (j < per && b0 + j < nbins) ? a[b0 + j] : 0u;
    s += v[j];
  }
  uint32_t ex = cta_exclusive_scan(s, scratch);
#pragma unroll
  for (int j = 0; j < kSortBinsPerThread; ++j) {
    if (j < per && b0 + j < nbins) a[b0 + j] = ex;
    ex += v[j];
  }
  __syncthreads();
}

// Add the digits of up to 32 elements (one per lane) to a shared-memory histogram.  A warp whose valid lanes
// all hold the same digit (heavy cell, or a nearly sorted input on a re-bin) adds once.
__device__ __forceinline__ void hist_add(uint32_t* h, uint32_t d, bool valid) {
  const uint32_t vm = __ballot_sync(0xffffffffu, valid);
  if (vm == 0u) return;
  const uint32_t d0 = __shfl_sync(0xffffffffu, d, __ffs(vm) - 1);
  if (__all_sync(0xffffffffu, !valid || d == d0)) {
    if ((threadIdx.x & 31) == 0) atomicAdd(&h[d0], (uint32_t)__popc(vm));
  } else if (valid) {
    atomicAdd(&h[d], 1u);
  }
}

// ------------------------------------------------- A1 + A2: cell ids, flags, first-digit histogram --
// Histograms are kept per TILE of 4096 consecutive elements (hist[tile][bin]); CTAs take tiles round-robin.
__global__ void __launch_bounds__(kSortThreads) k_keys_hist(const float4* __restrict__ pos_mass, int64_t n, Geometry g,
                                                             uint32_t* __restrict__ keys, DevFlags* flags, int nbins,
                                                             uint32_t* __restrict__ hist, int64_t ntiles) {
  extern __shared__ uint32_t h_dyn[];
  const float m0 = __ldg(&pos_mass[0].w);
  const uint32_t mask = (uint32_t)nbins - 1u;
  uint32_t bad = 0, mdiff = 0;
  for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
    for (int d = threadIdx.x; d < nbins; d += kSortThreads) h_dyn[d] = 0u;
    __syncthreads();
    const int64_t beg = t * kSortTile, end = min(n, beg + kSortTile);
    float4 p[kSortItems];
#pragma unroll
    for (int u = 0; u < kSortItems; ++u) {
      const int64_t i = beg + threadIdx.x + u * kSortThreads;
      p[u] = i < end ? __ldcs(&pos_mass[i]) : make_float4(0.f, 0.f, 0.f, m0);
    }
#pragma unroll
    for (int u = 0; u < kSortItems; ++u) {
      const int64_t i = beg + threadIdx.x + u * kSortThreads;
      const bool valid = i < end;
      const bool ok = (p[u].x >= 0.f) && (p[u].x < g.box[0]) && (p[u].y >= 0.f) && (p[u].y < g.box[1]) &&
                      (p[u].z >= 0.f) && (p[u].z < g.box[2]);
      // one IEEE multiply per axis (never contracted: there is nothing to fuse with), floor, clamp (R10)
      int cx = (int)floorf(__fmul_rn(p[u].x, g.inv_cell[0]));
      int cy = (int)floorf(__fmul_rn(p[u].y, g.inv_cell[1]));
      int cz = (int)floorf(__fmul_rn(p[u].z, g.inv_cell[2]));
      cx = min(cx, g.ncell[0] - 1);
      cy = min(cy, g.ncell[1] - 1);
      cz = min(cz, g.ncell[2] - 1);
      const uint32_t id =
          ok ? (uint32_t)cx + (uint32_t)g.ncell[0] * ((uint32_t)cy + (uint32_t)g.ncell[1] * (uint32_t)cz) : 0u;
      if (valid) keys[i] = id;
      bad |= (valid && !ok) ? 1u : 0u;
      mdiff |= (valid && p[u].w != m0) ? 1u : 0u;   // NaN mass counts as different
      hist_add(h_dyn, id & mask, valid);
    }
    __syncthreads();
    for (int d = threadIdx.x; d < nbins; d += kSortThreads) hist[(size_t)t * nbins + d] = h_dyn[d];
    __syncthreads();
  }
  if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) atomicOr(&flags->domain_error, 1u);
  if (__any_sync(0xffffffffu, mdiff) && (threadIdx.x & 31) == 0) atomicOr(&flags->mass_nonuniform, 1u);
}

// ------------------------------------------------------ A2 (later digits): per-tile digit histogram --
__global__ void __launch_bounds__(kSortThreads) k_digit_hist(const uint32_t* __restrict__ keys, int64_t n, int shift,
                                                              int nbins, uint32_t* __restrict__ hist, int64_t ntiles) {
  extern __shared__ uint32_t h_dyn[];                  // two histograms: tiles alternate, one barrier per tile
  const uint32_t mask = (uint32_t)nbins - 1u;
  uint32_t k[kSortItems];
  {
    const int64_t beg = (int64_t)blockIdx.x * kSortTile;
#pragma unroll
    for (int u = 0; u < kSortItems; ++u) {
      const int64_t i = beg + threadIdx.x + u * kSortThreads;
      k[u] = i < n ? __ldcs(&keys[i]) : 0u;
    }
  }
  for (int d = threadIdx.x; d < 2 * nbins; d += kSortThreads) h_dyn[d] = 0u;
  __syncthreads();
  int buf = 0;
  for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x, buf ^= 1) {
    uint32_t* h = h_dyn + buf * nbins;
    const int64_t beg = t * kSortTile, end = min(n, beg + kSortTile);
    uint32_t cur[kSortItems];
#pragma unroll
    for (int u = 0; u < kSortItems; ++u) cur[u] = k[u];
    // next tile's keys are in flight while this tile is counted
    {
      const int64_t nbeg = (t + gridDim.x) * kSortTile;
#pragma unroll
      for (int u = 0; u < kSortItems; ++u) {
        const int64_t i = nbeg + threadIdx.x + u * kSortThreads;
        k[u] = i < n ? __ldcs(&keys[i]) : 0u;
      }
    }
#pragma unroll
    for (int u = 0; u < kSortItems; ++u)
      hist_add(h, (cur[u] >> shift) & mask, beg + threadIdx.x + u * kSortThreads < end);
    __syncthreads();
    // write this tile's row and clear the buffer for the tile after next (the other buffer is already clear)
    for (int d = threadIdx.x; d < nbins; d += kSortThreads) {
      hist[(size_t)t * nbins + d] = h[d];
      h[d] = 0u;
    }
  }
}

// -------------------------------------------- A3: per-digit exclusive scan over tiles + digit totals --
// hist[tile][bin] -> exclusive prefix over tiles (in place); coltot[bin] = total of the bin.  The tiles are
// cut into kScanSlices slices; grid = (bins/32, slices); a CTA owns 32 bins x one slice, warp w a sub-slice,
// lane = bin, so every access is a 128-byte row segment.  Phase 1 writes the slice totals, phase 2 adds the
// totals of the earlier slices and rewrites its slice as exclusive prefixes.
constexpr int kScanSlices = 8;

__global__ void __launch_bounds__(1024) k_col_sum(const uint32_t* __restrict__ hist, int64_t ntiles, int nbins,
                                                   uint32_t* __restrict__ part /*[kScanSlices][nbins]*/) {
  __shared__ uint32_t sm[32][33];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int bin = blockIdx.x * 32 + lane;
  const int64_t per_slice = (ntiles + kScanSlices - 1) / kScanSlices;
  const int64_t s0 = min(ntiles, blockIdx.y * per_slice), s1 = min(ntiles, s0 + per_slice);
  const int64_t per = (s1 - s0 + 31) / 32;
  const int64_t b0 = min(s1, s0 + w * per), b1 = min(s1, b0 + per);
  uint32_t s = 0;
#pragma unroll 8
  for (int64_t b = b0; b < b1; ++b) s += __ldg(&hist[(size_t)b * nbins + bin]);
  sm[w][lane] = s;
  __syncthreads();
  if (w == 0) {
    uint32_t tot = 0;
#pragma unroll
    for (int ww = 0; ww < 32; ++ww) tot += sm[ww][lane];
    part[(size_t)blockIdx.y * nbins + bin] = tot;
  }
}

__global__ void __launch_bounds__(1024) k_col_scan(uint32_t* __restrict__ hist, int64_t ntiles, int nbins,
                                                    const uint32_t* __restrict__ part, uint32_t* __restrict__ coltot) {
  __shared__ uint32_t sm[32][33];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int bin = blockIdx.x * 32 + lane;
  const int64_t per_slice = (ntiles + kScanSlices - 1) / kScanSlices;
  const int64_t s0 = min(ntiles, blockIdx.y * per_slice), s1 = min(ntiles, s0 + per_slice);
  const int64_t per = (s1 - s0 + 31) / 32;
  const int64_t b0 = min(s1, s0 + w * per), b1 = min(s1, b0 + per);
  uint32_t s = 0;
#pragma unroll 8
  for (int64_t b = b0; b < b1; ++b) s += hist[(size_t)b * nbins + bin];
  sm[w][lane] = s;
  __syncthreads();
  uint32_t run = 0, total = 0;
  for (int y = 0; y < kScanSlices; ++y) {
    const uint32_t v = __ldg(&part[(size_t)y * nbins + bin]);
    if (y < (int)blockIdx.y) run += v;
    total += v;
  }
  for (int ww = 0; ww < w; ++ww) run += sm[ww][lane];
#pragma unroll 8
  for (int64_t b = b0; b < b1; ++b) {
    const uint32_t v = hist[(size_t)b * nbins + bin];
    hist[(size_t)b * nbins + bin] = run;
    run += v;
  }
  if (blockIdx.y == 0 && w == 0) coltot[bin] = total;
}

// ---------------------------------------------------------------------- A4: stable scatter of a digit --
// CTAs take tiles of 4096 consecutive elements round-robin.  Inside a tile, warp w owns elements
// [256w, 256w+256) in 8 steps of 32 consecutive elements, so (tile, warp, step, lane) order == input order;
// ranks are assigned in that order.  The tile is then re-ordered by digit in shared memory and written out as
// per-digit runs (consecutive threads -> consecutive addresses inside a run).  Round-robin matters: the runs
// that the concurrently running CTAs write for one digit are ADJACENT in memory (tiles t, t+1, ... of the same
// digit), so the partially covered 32-byte sectors at the ends of a short run are completed by a neighbouring
// CTA while they are still in L2 (a partial sector that reaches DRAM costs a read-modify-write).
// Dynamic shared memory:  base[nbins] | tstart[nbins] | union{ u16 wc[16][nbins], {float4 spos[4096],
// u32 sidx[4096], u32 skey[4096]} } | scan scratch[16].
__host__ __device__ inline size_t scatter_smem_bytes(int nbins) {
  const size_t wc = (size_t)kSortWarps * nbins * sizeof(unsigned short);
  const size_t stage = (size_t)kSortTile * (sizeof(float4) + 2 * sizeof(uint32_t));
  return 2 * (size_t)nbins * sizeof(uint32_t) + (wc > stage ? wc : stage) + kSortWarps * sizeof(uint32_t);
}

// L2 policies: the inputs of a pass are read exactly once (evict_first); its outputs are written as short
// per-digit runs that the NEXT tile of the same CTA extends, so a partially written 32-byte sector has to
// stay in L2 until it is complete (evict_last) -- an evicted partial sector costs a DRAM read-modify-write.
__device__ __forceinline__ uint64_t policy_evict_first() {
  uint64_t p; asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p)); return p;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
  uint64_t p; asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p)); return p;
}
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src, uint64_t pol) {
  asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src), "l"(pol) : "memory");
}
__device__ __forceinline__ void cp_async4(void* smem_dst, const void* gmem_src, uint64_t pol) {
  asm volatile("cp.async.ca.shared.global.L2::cache_hint [%0], [%1], 4, %2;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src), "l"(pol) : "memory");
}
__device__ __forceinline__ uint32_t ld_stream_u32(const uint32_t* p, uint64_t pol) {
  uint32_t v; asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.u32 %0, [%1], %2;" : "=r"(v) : "l"(p), "l"(pol)); return v;
}
__device__ __forceinline__ void st_keep_u32(uint32_t* p, uint32_t v, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.u32 [%0], %1, %2;" ::"l"(p), "r"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_keep_f4(float4* p, float4 v, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1,%2,%3,%4}, %5;" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "l"(pol) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() {
  asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
}

// Only the 4-byte keys pass through registers (next tile's keys are prefetched while this tile's payload is in
// flight); the payload goes global -> shared with cp.async straight to its digit-ordered slot, so two CTAs
// fit per SM and one CTA's ranking overlaps the other's memory phase.
// Lanes of the warp holding the same digit as this lane (valid lanes only).  One ballot per digit bit:
// MATCH.ANY gives the same mask in one instruction but it is issued through the MIO queue at a rate that
// made the ranking loop the bottleneck of the whole pass (ncu: short-scoreboard + MIO-throttle stalls).
__device__ __forceinline__ uint32_t digit_peers(uint32_t d, bool valid, int dbits) {
  uint32_t peers = __ballot_sync(0xffffffffu, valid);
  for (int b = 0; b < dbits; ++b) {
    const bool bit = (d >> b) & 1u;
    const uint32_t bal = __ballot_sync(0xffffffffu, bit);
    peers &= bit ? bal : ~bal;
  }
  return peers;
}

template <bool kIdentityIdx>
__global__ void __launch_bounds__(kSortThreads, 2) k_digit_scatter(
    const uint32_t* __restrict__ keys_in, const float4* __restrict__ pos_in, const uint32_t* __restrict__ idx_in,
    uint32_t* __restrict__ keys_out, float4* __restrict__ pos_out, uint32_t* __restrict__ idx_out, int64_t n, int shift,
    int nbins, const uint32_t* __restrict__ hist, const uint32_t* __restrict__ coltot, int64_t ntiles) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int dbits = 31 - __clz(nbins);
  uint32_t* base = (uint32_t*)smem_raw;                            // start of every digit in the output
  uint32_t* tstart = base + nbins;
  unsigned char* un = (unsigned char*)(tstart + nbins);
  unsigned short* wc = (unsigned short*)un;                        // [kSortWarps][nbins]
  float4* spos = (float4*)un;                                      // [kSortTile]
  uint32_t* sidx = (uint32_t*)(un + (size_t)kSortTile * sizeof(float4));
  uint32_t* skey = sidx + kSortTile;
  const size_t un_bytes = scatter_smem_bytes(nbins) - 2 * (size_t)nbins * sizeof(uint32_t) - kSortWarps * sizeof(uint32_t);
  uint32_t* scratch = (uint32_t*)(un + un_bytes);

  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const uint32_t lt_mask = (1u << lane) - 1u;
  const uint32_t mask = (uint32_t)nbins - 1u;
  const int ebase = w * (32 * kSortItems) + lane;
  const uint64_t pol_in = policy_evict_first(), pol_out = policy_evict_last();

  uint32_t key[kSortItems];
#pragma unroll
  for (int s = 0; s < kSortItems; ++s) {
    const int64_t i = (int64_t)blockIdx.x * kSortTile + ebase + s * 32;
    key[s] = i < n ? ld_stream_u32(&keys_in[i], pol_in) : 0u;
  }
  // start of every digit in the output: exclusive scan of the digit totals
  for (int d = threadIdx.x; d < nbins; d += kSortThreads) base[d] = coltot[d];
  __syncthreads();
  cta_scan_bins(base, nbins, scratch);

  for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
    const int64_t tile = t * kSortTile;
    const int tile_n = (int)min((int64_t)kSortTile, n - tile);
    uint32_t goff[kSortBinsPerThread];      // first: elements of the digit in earlier tiles
#pragma unroll
    for (int j = 0; j < kSortBinsPerThread; ++j) {
      const int d = threadIdx.x + j * kSortThreads;
      goff[j] = d < nbins ? __ldg(&hist[(size_t)t * nbins + d]) : 0u;
    }
    // ---- zero the per-warp digit counters (the sync also fences the previous tile's staging reads)
    __syncthreads();
    {
      uint4* z = (uint4*)wc;
      const int nz = kSortWarps * nbins * (int)sizeof(unsigned short) / 16;
      for (int q = threadIdx.x; q < nz; q += kSortThreads) z[q] = make_uint4(0u, 0u, 0u, 0u);
    }
    __syncthreads();
    // ---- stable ranks inside the warp's 256 elements
    unsigned short* mywc = wc + (size_t)w * nbins;
    uint32_t rank[kSortItems];
#pragma unroll
    for (int s = 0; s < kSortItems; ++s) {
      const bool valid = ebase + s * 32 < tile_n;
      const uint32_t d = (key[s] >> shift) & mask;
      const uint32_t peers = digit_peers(d, valid, dbits);
      const uint32_t prev = valid ? (uint32_t)mywc[d] : 0u;
      rank[s] = prev + (uint32_t)__popc(peers & lt_mask);
      __syncwarp();
      if (valid && lane == (__ffs(peers) - 1)) mywc[d] = (unsigned short)(prev + (uint32_t)__popc(peers));
      __syncwarp();
    }
    __syncthreads();
    // ---- per digit: exclusive prefix over the warps; tile count of the digit -> tstart (scanned next)
    {   // two adjacent digits per thread: one 32-bit access carries both u16 counters (counts <= 4096: no carry)
      uint32_t* wc32 = (uint32_t*)wc;
      const int half = nbins >> 1;
      for (int dp = threadIdx.x; dp < half; dp += kSortThreads) {
        uint32_t run = 0;
#pragma unroll
        for (int r = 0; r < kSortWarps; ++r) {
          const uint32_t c = wc32[(size_t)r * half + dp];
          wc32[(size_t)r * half + dp] = run;
          run += c;
        }
        tstart[2 * dp] = run & 0xffffu;
        tstart[2 * dp + 1] = run >> 16;
      }
    }
    __syncthreads();
    cta_scan_bins(tstart, nbins, scratch);
    // ---- position of every element in the digit-ordered tile (reuses rank[])
#pragma unroll
    for (int s = 0; s < kSortItems; ++s) {
      const uint32_t d = (key[s] >> shift) & mask;
      rank[s] += tstart[d] + (uint32_t)mywc[d];
    }
    // goff[d] = (start of the digit + elements of the digit in earlier tiles) - its start inside this tile
#pragma unroll
    for (int j = 0; j < kSortBinsPerThread; ++j) {
      const int d = threadIdx.x + j * kSortThreads;
      if (d < nbins) goff[j] += base[d] - tstart[d];
    }
    __syncthreads();      // wc and tstart are dead from here: staging aliases wc, goff reuses tstart
    // ---- payload: global -> its slot of the digit-ordered tile, asynchronously
#pragma unroll
    for (int s = 0; s < kSortItems; ++s) {
      const int e = ebase + s * 32;
      if (e < tile_n) {
        const int64_t i = tile + e;
        cp_async16(&spos[rank[s]], &pos_in[i], pol_in);
        if (kIdentityIdx) sidx[rank[s]] = (uint32_t)i; else cp_async4(&sidx[rank[s]], &idx_in[i], pol_in);
        skey[rank[s]] = key[s];
      }
    }
#pragma unroll
    for (int j = 0; j < kSortBinsPerThread; ++j) {
      const int d = threadIdx.x + j * kSortThreads;
      if (d < nbins) tstart[d] = goff[j];
    }
    // ---- prefetch the next tile's keys while the payload is in flight
#pragma unroll
    for (int s = 0; s < kSortItems; ++s) {
      const int64_t i = (t + gridDim.x) * kSortTile + ebase + s * 32;
      key[s] = i < n ? ld_stream_u32(&keys_in[i], pol_in) : 0u;
    }
    cp_async_wait_all();
    __syncthreads();
    // ---- write out per-digit runs
#pragma unroll
    for (int s = 0; s < kSortItems; ++s) {
      const int q = s * kSortThreads + threadIdx.x;
      if (q < tile_n) {
        const uint32_t k = skey[q];
        const uint32_t dst = tstart[(k >> shift) & mask] + (uint32_t)q;
        st_keep_f4(&pos_out[dst], spos[q], pol_out);
        st_keep_u32(&idx_out[dst], sidx[q], pol_out);
        st_keep_u32(&keys_out[dst], k, pol_out);
      }
    }
  }
}

// --------------------------------------------------------------- cell_start from run boundaries --
__global__ void __launch_bounds__(256) k_cell_start(const uint32_t* __restrict__ sorted_keys, int64_t n, int32_t ncells,
                                                     uint32_t* __restrict__ cell_start) {
  constexpr int U = 8;
  for (int64_t k0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * U; k0 < n; k0 += (int64_t)gridDim.x * blockDim.x * U) {
    // keys k0-1 .. k0+U-1 (k0 is a multiple of 8: two 16-byte loads + the predecessor)
    uint32_t key[U + 1];
    key[0] = k0 > 0 ? __ldg(&sorted_keys[k0 - 1]) : 0u;
    if (k0 + U <= n) {
      const uint4 a = __ldg((const uint4*)&sorted_keys[k0]), b = __ldg((const uint4*)&sorted_keys[k0 + 4]);
      key[1] = a.x; key[2] = a.y; key[3] = a.z; key[4] = a.w; key[5] = b.x; key[6] = b.y; key[7] = b.z; key[8] = b.w;
    } else {
#pragma unroll
      for (int u = 0; u < U; ++u) key[u + 1] = k0 + u < n ? __ldg(&sorted_keys[k0 + u]) : 0u;
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t k = k0 + u;
      if (k < n) {
        const int64_t prev = k > 0 ? (int64_t)key[u] : -1;
        // cells (prev, key] start at k: the first is `key` itself, the rest are empty cells before it
        for (int64_t c = prev + 1; c <= (int64_t)key[u + 1]; ++c) cell_start[c] = (uint32_t)k;
        if (k == n - 1)
          for (int64_t c = (int64_t)key[u + 1] + 1; c <= (int64_t)ncells; ++c) cell_start[c] = (uint32_t)n;
      }
    }
  }
}

// ------------------------------------------------------------------------------------ host launcher --
// Digit plan: the cell id has `bits` significant bits; passes = ceil(bits / 8), digits of equal width.
void plan_sort(int32_t ncells, int* passes, int* digit_bits) {
  int bits = kSortMinDigitBits;
  while (((int64_t)1 << bits) < (int64_t)ncells) ++bits;
  const int p = (bits + kSortMaxDigitBits - 1) / kSortMaxDigitBits;
  *passes = p;
  *digit_bits = (bits + p - 1) / p;
}

cudaError_t launch_build_mesh(srpp_ctx* c, const float4* pos_mass, int64_t n) {
  cudaStream_t st = c->stream;
  cudaError_t e;
  if ((e = cudaMemsetAsync(c->flags, 0, sizeof(DevFlags), st)) != cudaSuccess) return e;
  const int32_t ncells = c->geo.ncells;
  const int passes = c->sort_passes, dbits = c->sort_digit_bits, nbins = 1 << dbits;
  // the last pass writes into sorted/keys[f]/vals[f]; earlier passes alternate with the scratch set
  const int f = (passes - 1) & 1;
  c->perm = c->vals[f];
  c->sorted_keys = c->keys[f];
  if (n == 0) return cudaMemsetAsync(c->cell_start, 0, sizeof(uint32_t) * ((size_t)ncells + 1), st);
  if (c->timing) cudaEventRecord(c->ev[kEvMesh0], st);

  const size_t smem_scatter = scatter_smem_bytes(nbins);
  if (!c->sort_attr_set) {
    if ((e = cudaFuncSetAttribute(k_digit_scatter<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)scatter_smem_bytes(kSortMaxBins))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_digit_scatter<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)scatter_smem_bytes(kSortMaxBins))) != cudaSuccess) return e;
    int occ = 1;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_digit_scatter<false>, kSortThreads, smem_scatter)) != cudaSuccess) return e;
    c->sort_blocks_per_sm = std::max(1, std::min(occ, 2));
    c->sort_attr_set = true;
  }
  const int64_t tiles = (n + kSortTile - 1) / kSortTile;
  const int blocks = (int)std::min<int64_t>(tiles, (int64_t)c->num_sms * c->sort_blocks_per_sm);
  const int hblocks = (int)std::min<int64_t>(tiles, (int64_t)c->num_sms * 4);
  c->sort_blocks = blocks;

  const size_t smem_hist = (size_t)nbins * sizeof(uint32_t);
  // buffer set A = {keys[0], vals[0], pos A}, set B = {keys[1], vals[1], pos B}; pos of the final set is `sorted`
  float4* posbuf[2];
  posbuf[f] = c->sorted;
  posbuf[f ^ 1] = c->pos_tmp;
  k_keys_hist<<<hblocks, kSortThreads, smem_hist, st>>>(pos_mass, n, c->geo, c->keys_raw, c->flags, nbins, c->hist, tiles);
  const uint32_t* kin = c->keys_raw;
  const float4* pin = pos_mass;
  const uint32_t* iin = nullptr;
  for (int p = 0; p < passes; ++p) {
    const int shift = p * dbits;
    const int o = p & 1;
    if (p > 0) k_digit_hist<<<hblocks, kSortThreads, 2 * smem_hist, st>>>(kin, n, shift, nbins, c->hist, tiles);
    k_col_sum<<<dim3(nbins / 32, kScanSlices), 1024, 0, st>>>(c->hist, tiles, nbins, c->colpart);
    k_col_scan<<<dim3(nbins / 32, kScanSlices), 1024, 0, st>>>(c->hist, tiles, nbins, c->colpart, c->coltot);
    if (p == 0)
      k_digit_scatter<true><<<blocks, kSortThreads, smem_scatter, st>>>(kin, pin, iin, c->keys[o], posbuf[o], c->vals[o], n, shift, nbins, c->hist, c->coltot, tiles);
    else
      k_digit_scatter<false><<<blocks, kSortThreads, smem_scatter, st>>>(kin, pin, iin, c->keys[o], posbuf[o], c->vals[o], n, shift, nbins, c->hist, c->coltot, tiles);
    kin = c->keys[o]; pin = posbuf[o]; iin = c->vals[o];
  }
  const int grid_ew = (int)std::min<int64_t>((n + 2047) / 2048, (int64_t)c->num_sms * 8);
  k_cell_start<<<grid_ew, 256, 0, st>>>(c->sorted_keys, n, ncells, c->cell_start);
  c->launches += 1 + 4 * (uint64_t)passes;
  if (c->timing) { cudaEventRecord(c->ev[kEvMesh1], st); c->ev_mesh_valid = true; }
  return cudaGetLastError();
}

}  // namespace srpp
