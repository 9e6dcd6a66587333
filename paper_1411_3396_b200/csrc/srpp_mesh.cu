// srpp_mesh.cu -- chaining-mesh binning (steps A1-A4 of SURVEY.md 8(a)) for sm_100a.
//
// The mesh is a STABLE counting sort of the particles by linear cell id (readings R10-R12):
//   A1  cell id per particle, fp32:  c = min((int)floorf(x * inv), ncell-1), inv = (float)ncell/box
//   A2-A4 histogram / exclusive scan / stable scatter.  A cell id has up to 24 bits and single cells hold
//        millions of particles, so the counting sort is applied digit-wise, least significant digit first,
//        in digits of <= 8 bits (three passes cover the 2^24-cell limit), with the particle PAYLOAD carried
//        through every pass so that all global traffic is a coalesced stream.
//   cell_start = run boundaries of the sorted ids (= exclusive prefix sum of the cell histogram).
//
// Round-2 structure (one kernel per pass, no per-tile histogram arrays, no key arrays):
//   k_sort_prepass   one read of the positions: domain / mass flags (R13, R14) and the GLOBAL histogram of every digit
//                    (A2; <= 3 x 256 counters).  The cell id is never stored: each pass recomputes it from the
//                    position it carries (3 multiplies + floor, far below the memory time).
//   k_sort_pass      per digit: two CTAs of 512 threads per SM take tiles of 4096 consecutive elements in ticket order,
//                    every thread holding 8 elements in registers (requested one tile ahead; the tile gridDim.x
//                    tickets ahead is pulled into L2 by a TMA prefetch); stable ranks come from per-warp {peer mask,
//                    running count} tables in warp-major order (no atomic decides a position, so perm is
//                    reproducible and equals the oracle's stable counting sort); the exclusive prefix of every digit
//                    over the earlier tiles comes from a decoupled look-back over per-tile status words (A3:
//                    aggregate published right after the tile histogram, inclusive prefix after the look-back); the
//                    tile is re-ordered by digit in shared memory and leaves as per-digit runs -- TMA bulk stores, one
//                    per digit thread, in every pass but the last (equal masses), ordinary stores otherwise.
//                    Equal masses (every BASELINE.json config): the original index travels in the .w lane of the
//                    position (16 bytes per element and pass) and the mass is restored by the last pass; otherwise it
//                    travels in a separate array (20 bytes).  The last pass also writes perm and the sorted cell ids.
//   k_cell_start     run boundaries of the sorted ids.
// Algorithmic bytes per build: 52*N + 8*ncells.  Moved by this design for three passes with equal
// masses: 16 (prepass) + 32 + 32 + 40 + 4 = 124 bytes per particle (round 1: 172), all coalesced.
// Paper context: PAPER.md:63/65 (direct PP short-range solver inside the hand-over radius); the chaining
// mesh itself is named by BASELINE.json north_star.
#include <algorithm>
#include <type_traits>

#include "srpp_internal.cuh"

namespace srpp {

// ------------------------------------------------------------------------------ small helpers --
// Exclusive scan of one value per thread over a kThreads-wide CTA; `scratch` holds 32 words.
template <int kThreads>
__device__ __forceinline__ uint32_t cta_exclusive_scan(uint32_t v, uint32_t* scratch) {
  constexpr int kWarps = kThreads / 32;
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
    uint32_t w = lane < kWarps ? scratch[lane] : 0u;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t y = __shfl_up_sync(0xffffffffu, w, o);
      if (lane >= o) w += y;
    }
    if (lane < kWarps) scratch[lane] = w;   // inclusive over warps
  }
  __syncthreads();
  return (wid ? scratch[wid - 1] : 0u) + (x - v);
}

// In-place exclusive scan of a[0..nbins) in shared memory (nbins a power of two, 32 <= nbins <= kSortMaxBins <= kThreads).
template <int kThreads>
__device__ __forceinline__ void cta_scan_bins(uint32_t* a, int nbins, uint32_t* scratch) {
  const uint32_t v = (int)threadIdx.x < nbins ? a[threadIdx.x] : 0u;
  const uint32_t ex = cta_exclusive_scan<kThreads>(v, scratch);
  if ((int)threadIdx.x < nbins) a[threadIdx.x] = ex;
  __syncthreads();
}

// L2 policies: the inputs of a pass are read exactly once (evict_first); its outputs are written as short
// per-digit runs that a neighbouring tile extends, so a partially written 32-byte sector has to stay in L2
// until it is complete (evict_last) -- an evicted partial sector costs a DRAM read-modify-write.
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
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void st_keep_u32(uint32_t* p, uint32_t v, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.u32 [%0], %1, %2;" ::"l"(p), "r"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_keep_f4(float4* p, float4 v, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1,%2,%3,%4}, %5;" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "l"(pol) : "memory");
}
// TMA bulk store of one per-digit run, shared -> global (16-byte aligned, a multiple of 16 bytes), with an L2 policy
__device__ __forceinline__ void bulk_store(void* gmem_dst, const void* smem_src, uint32_t bytes, uint64_t pol) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;" ::"l"(gmem_dst),
               "r"((uint32_t)__cvta_generic_to_shared(smem_src)), "r"(bytes), "l"(pol) : "memory");
}
// TMA prefetch of a contiguous global range into L2 (no registers, no shared memory); bytes a multiple of 16
__device__ __forceinline__ void bulk_prefetch_l2(const void* gmem, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(gmem), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ unsigned long long ld_status(const unsigned long long* p) {
  unsigned long long v; asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory"); return v;
}
__device__ __forceinline__ void st_status(unsigned long long* p, unsigned long long v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// ------------------------------------------ A1 + A2: flags and the global histogram of every digit --
__global__ void __launch_bounds__(kSortThreads) k_sort_prepass(const float4* __restrict__ pos_mass, int64_t n, Geometry g,
                                                                DevFlags* flags, int passes, int dbits,
                                                                uint32_t* __restrict__ ghist /*[passes][kSortMaxBins]*/) {
  __shared__ uint32_t h[kSortMaxPasses * kSortMaxBins];
  const int nbins = 1 << dbits;
  const uint32_t mask = (uint32_t)nbins - 1u;
  for (int d = threadIdx.x; d < passes * kSortMaxBins; d += kSortThreads) h[d] = 0u;
  __syncthreads();
  const uint32_t m0 = __float_as_uint(__ldg(&pos_mass[0].w));
  uint32_t bad = 0, mdiff = 0;
  const int64_t ntiles = (n + kSortTile - 1) / kSortTile;
  for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
    const int64_t beg = t * kSortTile, end = min(n, beg + kSortTile);
    float4 p[kSortItems];
#pragma unroll
    for (int u = 0; u < kSortItems; ++u) {
      const int64_t i = beg + threadIdx.x + u * kSortThreads;
      p[u] = i < end ? __ldcs(&pos_mass[i]) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
#pragma unroll
    for (int u = 0; u < kSortItems; ++u) {
      const bool valid = beg + threadIdx.x + u * kSortThreads < end;
      const uint32_t id = cell_key(p[u], g);
      bad |= (valid && !in_domain(p[u], g)) ? 1u : 0u;
      mdiff |= (valid && __float_as_uint(p[u].w) != m0) ? 1u : 0u;   // bitwise: the packed path restores m0's bits
      // one shared-memory atomic per digit; a warp whose lanes all hold the same cell (a heavy cell in a nearly
      // sorted input: 32-way same-address serialisation otherwise) adds once per digit instead
      const uint32_t vm = __ballot_sync(0xffffffffu, valid);
      const uint32_t id0 = __shfl_sync(0xffffffffu, id, vm ? __ffs(vm) - 1 : 0);
      const bool same = __all_sync(0xffffffffu, !valid || id == id0);
      if (same) {
        if ((threadIdx.x & 31) == 0 && vm)
          for (int q = 0; q < passes; ++q) atomicAdd(&h[q * kSortMaxBins + ((id0 >> (q * dbits)) & mask)], (uint32_t)__popc(vm));
      } else if (valid) {
        for (int q = 0; q < passes; ++q) atomicAdd(&h[q * kSortMaxBins + ((id >> (q * dbits)) & mask)], 1u);
      }
    }
  }
  __syncthreads();
  for (int d = threadIdx.x; d < passes * kSortMaxBins; d += kSortThreads)
    if (h[d]) atomicAdd(&ghist[d], h[d]);
  if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) atomicOr(&flags->domain_error, 1u);
  if (__any_sync(0xffffffffu, mdiff) && (threadIdx.x & 31) == 0) atomicOr(&flags->mass_nonuniform, 1u);
}

// ---------------------------------------------------------------------- A3 + A4: one digit pass --
// Per-tile status word of the decoupled look-back: high 32 bits = tag (epoch << 2 | kind), low 32 bits = count.
// kind 1: the tile's own count of the digit (aggregate); kind 2: inclusive prefix over tiles 0..t.  The epoch
// changes with every pass of every build, so the array never needs clearing between passes.
constexpr uint32_t kStatAgg = 1u, kStatPrefix = 2u;
#ifndef SRPP_PASS_THREADS
#define SRPP_PASS_THREADS 512
#endif
#ifndef SRPP_PASS_CTAS
#define SRPP_PASS_CTAS 2
#endif
#ifndef SRPP_L2_PREFETCH
#define SRPP_L2_PREFETCH 1
#endif
#ifndef SRPP_BULK_STORE
#define SRPP_BULK_STORE 1
#endif
#ifndef SRPP_LOOK_WINDOW
#define SRPP_LOOK_WINDOW 4
#endif
// Two CTAs of 512 threads per SM, 8 elements per thread: a pass is bound by issue slots, shared-memory wavefronts and
// the barrier-separated phases of a tile, not by DRAM, and the second CTA fills the first one's barrier waits
// (measured on config 4: 1024 threads x 1 CTA 1.38 ms per build, 512 x 2 1.25 ms; tiles of 2048 elements are slower:
// shorter per-digit runs).  The tunables can be overridden with -D for experiments.
constexpr int kPassThreads = SRPP_PASS_THREADS;
constexpr int kPassWarps = kPassThreads / 32;
constexpr int kPassItems = kPassTile / kPassThreads;
constexpr int kPassCtasPerSm = SRPP_PASS_CTAS;
constexpr int kLookWindow = SRPP_LOOK_WINDOW;                          // status words of earlier tiles read per round trip

// Dynamic shared memory of a pass (bytes), for nbins bins.
__host__ __device__ inline size_t sort_pass_smem(int nbins, bool packed) {
  size_t b = (size_t)kPassTile * sizeof(float4);                          // tile in digit order
  if (!packed) b += (size_t)kPassTile * sizeof(uint32_t);                 // original indices in digit order
  b += 2 * (size_t)kPassWarps * nbins * sizeof(uint32_t);                 // per-warp peer masks and counts per digit
  b += 3 * (size_t)nbins * sizeof(uint32_t);                              // base, tstart, goff
  b += 64 * sizeof(uint32_t);                                             // warp sums + tickets
  return b;
}

// One digit pass.  Per tile of 4096 consecutive elements (ticket order):
//   * every thread holds kPassItems (8) elements of the tile in registers (warp w owns the 256 consecutive elements
//     [256 w, 256 w + 256) in 8 steps of 32, so (tile, warp, step, lane) order == input order); they were requested
//     as soon as the previous tile had left the registers;
//   * stable ranks, no atomic decides a position: per step the lanes holding the same digit find each other through a
//     per-warp table -- every lane ORs its lane bit into the mask of its digit, reads mask and running count back
//     (rank = count + number of lower peers), and the lowest peer clears the mask and advances the count.  Which
//     lane's OR lands first does not matter: the mask is a set.  (Round 1 searched the peers with one ballot per digit
//     bit, about 40 instructions per step.)
//   * digit threads: exclusive prefix over the warps, tile count -> aggregate published for the look-back ->
//     exclusive scan over the digits (warp shuffles + one named barrier among the digit threads) -> decoupled
//     look-back over the earlier tiles' status words, kLookWindow of them per round trip;
//   * the elements go to their slot of the digit-ordered tile in shared memory and are written out as per-digit runs,
//     consecutive threads -> consecutive addresses (stores of single 16-byte elements straight to their final place
//     were measured at a third of this speed).  Four CTA barriers per tile.
// kBulk (equal masses, every pass but the last): the per-digit runs of the digit-ordered tile leave shared memory as
// TMA bulk stores, one per digit thread (cp.async.bulk: 128 runs of ~512 bytes per tile reach the HBM write rate,
// measured), so the write-out phase and its barrier disappear: a tile is rank -> scan -> slot store + look-back ->
// issue, three barriers, and the stores drain while the next tile is ranked.
template <bool kPacked, bool kBulk>
__global__ void __launch_bounds__(kPassThreads, kPassCtasPerSm) k_sort_pass(
    const float4* __restrict__ pos_in, const uint32_t* __restrict__ idx_in, float4* __restrict__ pos_out,
    uint32_t* __restrict__ idx_out, uint32_t* __restrict__ keys_out, const float4* __restrict__ pos_orig, int64_t n,
    Geometry g, int shift, int nbins, int first, int last, const uint32_t* __restrict__ ghist,
    unsigned long long* __restrict__ status, uint32_t* __restrict__ ticket, uint32_t epoch,
    const DevFlags* __restrict__ flags) {
  // the mode is a device-side fact (found by the prepass): both instantiations are launched, one returns at once
  if ((flags->mass_nonuniform == 0u) != kPacked) return;
  static_assert(!kBulk || kPacked, "bulk stores carry whole 16-byte elements");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float4* spos = (float4*)smem_raw;                                        // [kPassTile] digit order
  uint32_t* sidx = (uint32_t*)(spos + kPassTile);                          // [kPassTile]   (!kPacked only)
  uint32_t* masks = sidx + (kPacked ? 0 : kPassTile);                      // [kPassWarps][nbins]
  uint32_t* counts = masks + (size_t)kPassWarps * nbins;                   // [kPassWarps][nbins]
  uint32_t* base = counts + (size_t)kPassWarps * nbins;                    // start of every digit in the output
  uint32_t* tstart = base + nbins;                                         // start of every digit inside the tile
  uint32_t* goff = tstart + nbins;                                         // global start of the digit's run - tstart
  uint32_t* scratch = goff + nbins;                                        // [32] warp sums, [32..] tickets

  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const uint32_t lt_mask = (1u << lane) - 1u;
  const uint32_t mask = (uint32_t)nbins - 1u;
  const int ebase = w * (32 * kPassItems) + lane;
  const uint64_t pol_out = policy_evict_last();
  const int64_t ntiles = (n + kPassTile - 1) / kPassTile;
  const unsigned long long tag_agg = ((unsigned long long)((epoch << 2) | kStatAgg)) << 32;
  const unsigned long long tag_pre = ((unsigned long long)((epoch << 2) | kStatPrefix)) << 32;
  const uint32_t m0 = __float_as_uint(__ldg(&pos_orig[0].w));
  uint32_t* mymask = masks + (size_t)w * nbins;
  uint32_t* mycount = counts + (size_t)w * nbins;

  // start of every digit in the output: exclusive scan of the digit totals; clear the peer masks once (the leaders
  // leave them clear)
  if ((int)threadIdx.x < nbins) base[threadIdx.x] = ghist[threadIdx.x];
  for (int q = threadIdx.x; q < kPassWarps * nbins; q += kPassThreads) masks[q] = 0u;
  // Tiles are taken in ticket order, one ahead (a ticket held longer would stall the look-back of every later tile).
  // The tile a CTA will take after the next one is, in the steady state, about gridDim.x tickets further on: that
  // tile is pulled into L2 by one TMA prefetch, so that the register loads of whichever CTA gets it find it there.
  auto prefetch_tile = [&](int64_t tile) {
    if (SRPP_L2_PREFETCH && tile < ntiles) {
      const int64_t cnt = min((int64_t)kPassTile, n - tile * kPassTile);
      bulk_prefetch_l2(pos_in + tile * kPassTile, (uint32_t)cnt * (uint32_t)sizeof(float4));
      if (!kPacked && !first) bulk_prefetch_l2(idx_in + tile * kPassTile, (uint32_t)((cnt * 4 + 15) & ~15ll));
    }
  };
  if (threadIdx.x == 0) {
    const uint32_t t0 = atomicAdd(ticket, 1u);
    scratch[32] = t0;
    prefetch_tile((int64_t)t0 + gridDim.x);
  }
  __syncthreads();
  cta_scan_bins<kPassThreads>(base, nbins, scratch);
  int64_t t = scratch[32];

  // the tile's elements live in registers from the load to the slot store; the next tile is requested while this
  // one is written out.  (Addresses are clamped instead of predicated: a predicated load with a default value needs a
  // select right behind it, which makes the warp wait for the data at once.)
  float4 p[kPassItems];
  uint32_t ix[kPassItems];
  auto load_tile = [&](int64_t tile) {
    const int64_t tb = min(tile, ntiles - 1) * kPassTile;
#pragma unroll
    for (int s = 0; s < kPassItems; ++s) {
      const int64_t i = min(tb + ebase + s * 32, n - 1);
      p[s] = __ldcs(&pos_in[i]);
      if (!kPacked && !first) ix[s] = __ldcs(&idx_in[i]);
    }
  };
  load_tile(t);

  while (t < ntiles) {
    const int64_t tile = t * kPassTile;
    const int tile_n = (int)min((int64_t)kPassTile, n - tile);
    if (threadIdx.x == 0) {
      const uint32_t tn = atomicAdd(ticket, 1u);
      scratch[33] = tn;
      prefetch_tile((int64_t)tn + gridDim.x);
    }
    for (int q = lane; q < nbins; q += 32) mycount[q] = 0u;
    __syncwarp();
    // ---- stable ranks inside the warp's 128 consecutive elements
    uint32_t rd[kPassItems];            // rank | digit << 16
#pragma unroll
    for (int s = 0; s < kPassItems; ++s) {
      const bool valid = ebase + s * 32 < tile_n;
      const uint32_t d = (cell_key(p[s], g) >> shift) & mask;
      if (valid) atomicOr(&mymask[d], 1u << lane);
      __syncwarp();
      const uint32_t peers = mymask[d], prev = mycount[d];
      rd[s] = (prev + (uint32_t)__popc(peers & lt_mask)) | (d << 16);
      __syncwarp();
      if (valid && (peers & lt_mask) == 0u) { mymask[d] = 0u; mycount[d] = prev + (uint32_t)__popc(peers); }
      __syncwarp();
    }
    __syncthreads();                                     // B1: all tables complete; ticket visible
    const int64_t t_next = scratch[33];
    // ---- digit threads: prefix over the warps, tile count, aggregate, scan over the digits
    uint32_t cnt_keep = 0, ts_keep = 0;
    if ((int)threadIdx.x < nbins) {
      const int d = threadIdx.x;
      uint32_t run = 0;
#pragma unroll 1
      for (int r0 = 0; r0 < kPassWarps; r0 += 4) {
        uint32_t cnt[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) cnt[r] = counts[(size_t)(r0 + r) * nbins + d];     // four loads in flight at once
#pragma unroll
        for (int r = 0; r < 4; ++r) {
          counts[(size_t)(r0 + r) * nbins + d] = run;
          run += cnt[r];
        }
      }
      const uint32_t cnt_d = run;
      st_status(&status[(size_t)t * nbins + d], (t == 0 ? tag_pre : tag_agg) | cnt_d);
      // exclusive scan of the tile counts over the digits: warp scan + sums of the earlier digit warps
      uint32_t x = cnt_d;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
      }
      if (lane == 31) scratch[w] = x;
      asm volatile("bar.sync 1, %0;" ::"r"(nbins) : "memory");      // named barrier among the digit threads only
      uint32_t off = 0;
      for (int r = 0; r < w; ++r) off += scratch[r];
      const uint32_t ts = off + x - cnt_d;
      tstart[d] = ts;
      cnt_keep = cnt_d; ts_keep = ts;
      if (kBulk) bulk_wait_read();                       // the previous tile's runs have left shared memory
    }
    __syncthreads();                                     // B2: tstart and the prefixes over the warps are ready
    // ---- every element to its slot of the digit-ordered tile
#pragma unroll
    for (int s = 0; s < kPassItems; ++s) {
      const int e = ebase + s * 32;
      if (e < tile_n) {
        const uint32_t d = rd[s] >> 16;
        const uint32_t slot = tstart[d] + mycount[d] + (rd[s] & 0xffffu);
        uint32_t idx;
        if (first) idx = (uint32_t)(tile + e);
        else if (kPacked) idx = __float_as_uint(p[s].w);
        else idx = ix[s];
        float4 v = p[s];
        if (kPacked) v.w = __uint_as_float(idx); else sidx[slot] = idx;
        spos[slot] = v;
      }
    }
    if (kBulk) {
      fence_async_smem();                                // the slot stores become visible to the TMA engine
      load_tile(t_next);                                 // registers are free again: request the next tile now
    }
    // ---- digit threads: decoupled look-back (the other warps are storing their elements meanwhile)
    if ((int)threadIdx.x < nbins) {
      const int d = threadIdx.x;
      uint32_t excl = 0;                                 // elements of the digit in tiles 0..t-1
      if (t > 0) {
        int64_t tt = t - 1;
        bool done = false;
        while (!done) {
          unsigned long long sw[kLookWindow];
#pragma unroll
          for (int j = 0; j < kLookWindow; ++j) sw[j] = tt - j >= 0 ? ld_status(&status[(size_t)(tt - j) * nbins + d]) : 0ull;
#pragma unroll
          for (int j = 0; j < kLookWindow; ++j) {
            if (done || tt - j < 0) continue;
            if (((uint32_t)(sw[j] >> 34)) != (epoch & 0x3fffffffu)) { tt -= j; goto again; }   // not published yet: re-poll from here
            excl += (uint32_t)sw[j];
            if ((((uint32_t)(sw[j] >> 32)) & 3u) == kStatPrefix) done = true;
          }
          tt -= kLookWindow;
        again:;
        }
        st_status(&status[(size_t)t * nbins + d], tag_pre | (unsigned long long)(excl + cnt_keep));
      }
      goff[d] = base[d] + excl - ts_keep;
    }
    __syncthreads();                                     // B3: digit-ordered tile and goff complete
    if (kBulk) {
      if ((int)threadIdx.x < nbins) {
        if (cnt_keep) bulk_store(pos_out + goff[threadIdx.x] + ts_keep, spos + ts_keep, cnt_keep * (uint32_t)sizeof(float4), pol_out);
        bulk_commit();
      }
      t = t_next;
      continue;                                          // no fourth barrier: see the reuse notes above each structure
    }
    // ---- next tile's elements are requested now, this tile is written out as per-digit runs meanwhile
    load_tile(t_next);
#pragma unroll
    for (int s = 0; s < kPassItems; ++s) {
      const int q = s * kPassThreads + threadIdx.x;
      if (q < tile_n) {
        float4 v = spos[q];
        // the digit is recomputed from the position: the ALUs idle while shared memory is the busy unit of this kernel
        const uint32_t key = cell_key(v, g);
        const uint32_t dst = goff[(key >> shift) & mask] + (uint32_t)q;
        if (last) {
          st_keep_u32(&keys_out[dst], key, pol_out);
          st_keep_u32(&idx_out[dst], kPacked ? __float_as_uint(v.w) : sidx[q], pol_out);
          if (kPacked) v.w = __uint_as_float(m0);
        } else if (!kPacked) {
          st_keep_u32(&idx_out[dst], sidx[q], pol_out);
        }
        st_keep_f4(&pos_out[dst], v, pol_out);
      }
    }
    t = t_next;
    __syncthreads();                                     // B4: the digit-ordered tile, goff and the ticket word are reused
  }
  if (kBulk && (int)threadIdx.x < nbins) bulk_wait_all();
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

// Stable sort of n particles by cell id into the buffers of `sb` (the context's own for srpp_build_mesh, a second set
// for the movers of the incremental re-bin): sb.out_sorted / sb.perm / sb.keys_out / sb.cell_start.
cudaError_t sort_by_cell(srpp_ctx* c, SortBufs& sb, const float4* pos_mass, int64_t n) {
  cudaStream_t st = c->stream;
  cudaError_t e;
  if ((e = cudaMemsetAsync(sb.flags, 0, sizeof(DevFlags), st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(sb.ctl, 0, sort_ctl_bytes(), st)) != cudaSuccess) return e;
  const int32_t ncells = c->geo.ncells;
  const int passes = c->sort_passes, dbits = c->sort_digit_bits, nbins = 1 << dbits;
  // the last pass writes into out_sorted / vals[f]; earlier passes alternate with the scratch set
  const int f = (passes - 1) & 1;
  sb.perm = sb.vals[f];
  if (n == 0) return cudaMemsetAsync(sb.cell_start, 0, sizeof(uint32_t) * ((size_t)ncells + 1), st);

  const size_t smem_packed = sort_pass_smem(nbins, true), smem_plain = sort_pass_smem(nbins, false);
  if (!c->sort_attr_set) {
    if ((e = cudaFuncSetAttribute(k_sort_pass<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sort_pass_smem(kSortMaxBins, true))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_sort_pass<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sort_pass_smem(kSortMaxBins, true))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_sort_pass<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sort_pass_smem(kSortMaxBins, false))) != cudaSuccess) return e;
    c->sort_attr_set = true;
  }
  const int64_t tiles = (n + kSortTile - 1) / kSortTile, ptiles = (n + kPassTile - 1) / kPassTile;
  // the look-back status words are tagged with an epoch, so they are cleared only when the array moves, grows, or
  // the epoch counter wraps (tags of another layout / an earlier life of the workspace must not be mistaken for ours)
  if (c->sort_epoch > 0x3ffffff0u) { c->sort_epoch = 0; c->status_n = 0; c->status_n_movers = 0; }
  if (*sb.status_n < n || *sb.status_n == 0) {
    if ((e = cudaMemsetAsync(sb.status, 0, sizeof(unsigned long long) * (size_t)ptiles * kSortMaxBins, st)) != cudaSuccess) return e;
    *sb.status_n = n;
  }
  const int blocks = (int)std::min<int64_t>(ptiles, (int64_t)c->num_sms * kPassCtasPerSm);
  const int hblocks = (int)std::min<int64_t>(tiles, (int64_t)c->num_sms * 2);

  uint32_t* tickets = sb.ctl;
  uint32_t* ghist = sb.ctl + 64;
  float4* posbuf[2];
  posbuf[f] = sb.out_sorted;
  posbuf[f ^ 1] = sb.tmp_pos;
  k_sort_prepass<<<hblocks, kSortThreads, 0, st>>>(pos_mass, n, c->geo, sb.flags, passes, dbits, ghist);
  const float4* pin = pos_mass;
  const uint32_t* iin = nullptr;
  for (int p = 0; p < passes; ++p) {
    const int shift = p * dbits;
    const int o = p & 1;
    const int first = p == 0, last = p == passes - 1;
    const uint32_t epoch = ++c->sort_epoch;
    if (SRPP_BULK_STORE && !last)
      k_sort_pass<true, true><<<blocks, kPassThreads, smem_packed, st>>>(pin, iin, posbuf[o], sb.vals[o], sb.keys_out, pos_mass, n, c->geo, shift, nbins, first, last, ghist + (size_t)p * kSortMaxBins, sb.status, tickets + p, epoch, sb.flags);
    else
      k_sort_pass<true, false><<<blocks, kPassThreads, smem_packed, st>>>(pin, iin, posbuf[o], sb.vals[o], sb.keys_out, pos_mass, n, c->geo, shift, nbins, first, last, ghist + (size_t)p * kSortMaxBins, sb.status, tickets + p, epoch, sb.flags);
    k_sort_pass<false, false><<<blocks, kPassThreads, smem_plain, st>>>(pin, iin, posbuf[o], sb.vals[o], sb.keys_out, pos_mass, n, c->geo, shift, nbins, first, last, ghist + (size_t)p * kSortMaxBins, sb.status, tickets + p, epoch, sb.flags);
    pin = posbuf[o]; iin = sb.vals[o];
  }
  const int grid_ew = (int)((n + 2047) / 2048);     // one trip per thread: the loads of all CTAs overlap
  k_cell_start<<<grid_ew, 256, 0, st>>>(sb.keys_out, n, ncells, sb.cell_start);
  c->launches += 2 + 2 * (uint64_t)passes;
  return cudaGetLastError();
}

cudaError_t launch_build_mesh(srpp_ctx* c, const float4* pos_mass, int64_t n) {
  cudaStream_t st = c->stream;
  if (c->timing && n > 0) cudaEventRecord(c->ev[kEvMesh0], st);
  // a full build always lands in the primary buffers (the incremental re-bin of srpp_subcycle ping-pongs)
  SortBufs sb;
  sb.flags = c->flags; sb.ctl = c->sort_ctl; sb.status = c->sort_status; sb.status_n = &c->status_n;
  sb.out_sorted = c->sorted_buf[0]; sb.tmp_pos = c->pos_tmp; sb.vals[0] = c->vals[0]; sb.vals[1] = c->vals[1];
  sb.keys_out = c->keys_buf[0]; sb.cell_start = c->cell_start; sb.perm = nullptr;
  const cudaError_t e = sort_by_cell(c, sb, pos_mass, n);
  if (e != cudaSuccess) return e;
  c->sorted = c->sorted_buf[0];
  c->sorted_keys = c->keys_buf[0];
  c->perm = sb.perm;
  if (c->timing && n > 0) { cudaEventRecord(c->ev[kEvMesh1], st); c->ev_mesh_valid = true; }
  return cudaGetLastError();
}

}  // namespace srpp
