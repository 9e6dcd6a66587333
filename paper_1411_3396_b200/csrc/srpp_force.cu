// srpp_force.cu -- short-range PP force (A5), write-back (A6), kick (A7) and stream for sm_100a.
//
//   a_i = sum_{j, s_ij < rc^2} m_j d_ij [ (s_ij + eps^2)^(-3/2) - P(s_ij) ]          (
//                                                                                    PAPER.md:63,65)
// Design:
//   * Work item = (cell c, tile of <= 32*T consecutive sorted targets of c, chunk of <= 1024 consecutive
//     positions of c's 27-cell source stream).  Items of all cells form one global index space
//     (exclusive prefix over cells); autonomous WARPS pull item indices from one atomic counter, so a
//     cell holding 600 k particles becomes ~10^6 small items spread over the whole chip -- the on-chip
//     analogue of the paper's block splitting for load balance.
//   * Targets live in registers as PACKED PAIRS (float2 = two targets); sources are staged by the warp into a
//     private shared-memory tile of float4 (x, y, z, m), read with one LDS.128 per source and fed to the packed
//     instructions as broadcast operands, so that every arithmetic instruction of the pair loop is a Blackwell
//     packed-fp32 op (FFMA2/FADD2/FMUL2): 16 packed FMA-pipe instructions per two pair interactions, leaving
//     issue slots for MUFU.RSQ and the cutoff select.
//   * Periodic images are applied when a source segment is staged (a per-segment shift), never per pair.
//     Staged coordinates are relative to integer reference points, so the wrap is exact in fp32.
//   * u = s + eps^2 comes straight out of the FMA chain (seeded with eps^2); the grid-force polynomial
//     is re-expanded in u on the host in fp64 (Q(u) = P(u - eps^2)), negated, so f = fma(r^2, r, -Q(u)).
//   * Each item accumulates in fp32 from zero over <= 1024 sources and is folded into fp64 accumulators
//     with red.global.add.f64; A6 converts to fp32 and writes in the caller's original order (R15).
#include <algorithm>

#include "srpp_internal.cuh"

namespace srpp {

// ------------------------------------------------------------------------------ stencil segments --
// The 27-cell stencil of cell (cx,cy,cz) as <= 18 runs that are contiguous in sorted order: 9 (dy,dz)
// rows x {main x-run, wrapped x-run}.  shift = periodic image offset to ADD to a source coordinate.
struct Segment {
  uint32_t start, end;      // sorted-index range
  int xlo, cy, cz;          // first cell of the run (for the reference point)
  float shift[3];
};

__device__ __forceinline__ Segment stencil_segment(const Geometry& g, const uint32_t* __restrict__ cell_start, int cx,
                                                   int cy, int cz, int seg) {
  Segment s;
  const int row = seg >> 1, sx = seg & 1;
  const int dy = row % 3 - 1, dz = row / 3 - 1;
  int y = cy + dy, z = cz + dz;
  s.shift[0] = 0.f; s.shift[1] = 0.f; s.shift[2] = 0.f;
  bool empty = false;
  if (y < 0) { y += g.ncell[1]; s.shift[1] = -g.box[1]; empty |= !g.periodic[1]; }
  else if (y >= g.ncell[1]) { y -= g.ncell[1]; s.shift[1] = g.box[1]; empty |= !g.periodic[1]; }
  if (z < 0) { z += g.ncell[2]; s.shift[2] = -g.box[2]; empty |= !g.periodic[2]; }
  else if (z >= g.ncell[2]) { z -= g.ncell[2]; s.shift[2] = g.box[2]; empty |= !g.periodic[2]; }
  const int ncx = g.ncell[0];
  int xlo, xhi;  // inclusive; xhi < xlo means empty
  if (cx >= 1 && cx <= ncx - 2) {
    if (sx == 0) { xlo = cx - 1; xhi = cx + 1; } else { xlo = 0; xhi = -1; }
  } else if (cx == 0) {
    if (sx == 0) { xlo = ncx - 1; xhi = g.periodic[0] ? ncx - 1 : ncx - 2; s.shift[0] = -g.box[0]; } else { xlo = 0; xhi = 1; }
  } else {
    if (sx == 0) { xlo = ncx - 2; xhi = ncx - 1; } else { xlo = 0; xhi = g.periodic[0] ? 0 : -1; s.shift[0] = g.box[0]; }
  }
  if (empty) xhi = xlo - 1;   // the (dy,dz) row lies beyond an open face
  s.xlo = xlo; s.cy = y; s.cz = z;
  if (xhi < xlo) { s.start = 0; s.end = 0; return s; }
  const int rowbase = ncx * (y + g.ncell[1] * z);
  s.start = __ldg(&cell_start[rowbase + xlo]);
  s.end = __ldg(&cell_start[rowbase + xhi + 1]);
  return s;
}

// Targets of one work item.  Large cells: 32 lanes x 8 targets (four packed pairs per lane), several items per cell.
// Cells of <= 48 particles (the uniform background: ~33 per cell) would leave half of a 64-target tile empty, so
// there the warp is split over the SOURCES: with S source phases, 32/S lanes x 2 targets = 64/S targets per packed
// pair, TP packed pairs per lane cover the WHOLE cell in one item (the staged sources are shared by all its targets),
// lane group g = lane / (32/S) takes sources g, g+S, g+2S, ... of the staged tile, and the S partial sums are added
// with shuffles at the end.  Cells of <= 40 particles use S = 8 (targets padded to a multiple of 8: 1.10 pair slots
// per candidate pair at ~33 per cell; S = 4 with its multiples of 16 gave 1.23), 41..48 use S = 4 (48 slots), 49..64
// take one 64-target item.
// Two builds of the force kernel; the plan kernel decides on the device which one runs (the other returns at once):
//   build 0 (most of W in cells of <= 64 particles: the uniform background, configs 1-2): CTAs of 8 warps, 2 per SM
//            = 16 warps with <= 128 registers -- the small-cell items are short and latency-bound, more warps win
//            (config 2: 55.9 % of FP32 peak against 53.6 % with build 1);
//   build 1 (most of W in large cells: every clustered config): CTAs of 4 warps, 3 per SM = 12 warps with <= 168
//            registers, which the large-cell item needs for its 4 packed target pairs per lane (256 targets) and 8
//            sources per trip (config 3: 74.8 % of FP32 peak; with 128 registers the best form is 3 pairs x 16 sources
//            at 73.9 %, 4 pairs x 8 sources 72.4 %; 8 warps per SM with 212 / 251 registers and 6 / 8 pairs: 73.0 / 72.9 %).
// The work plan (items per cell) is the same for both: large-cell items hold kBigTP packed pairs per lane.
template <int kBuild> struct PPBuild;
template <> struct PPBuild<0> { static constexpr int kThreads = 256, kCtasPerSm = 2; };
template <> struct PPBuild<1> { static constexpr int kThreads = 128, kCtasPerSm = 3; };
constexpr int kBigTP = 4;                       // packed target pairs per lane of a large-cell item (256 targets per item)
constexpr uint32_t kSplit8MaxCell = 40;         // <= 5 packed pairs of 8 targets
constexpr uint32_t kSplitMaxCell = 48;          // <= 3 packed pairs of 16 targets
__device__ __forceinline__ uint32_t targets_per_item(uint32_t n_c, int fine) {
  if (n_c <= kSplit8MaxCell) return fine ? min(16u, ((n_c + 7u) / 8u) * 8u) : ((n_c + 7u) / 8u) * 8u;   // fine: tiny problems need more items
  if (n_c <= kSplitMaxCell) return fine ? 16u : 48u;
  return n_c <= 64u ? 64u : 64u * (uint32_t)kBigTP;
}

// ------------------------------------------------------------------- plan: items per cell, W, max --
__global__ void __launch_bounds__(256) k_plan_items(const uint32_t* __restrict__ cell_start, Geometry g, int fine,
                                                     unsigned long long* __restrict__ items, DevFlags* flags) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  unsigned long long w = 0, slots = 0, wbig = 0;
  uint32_t nmax = 0;
  if (c < g.ncells) {
    const uint32_t n_c = __ldg(&cell_start[c + 1]) - __ldg(&cell_start[c]);
    unsigned long long it = 0;
    const int cx = c % g.ncell[0], cy = (c / g.ncell[0]) % g.ncell[1], cz = c / (g.ncell[0] * g.ncell[1]);
    const bool active = cx >= g.act_lo[0] && cx < g.act_hi[0] && cy >= g.act_lo[1] && cy < g.act_hi[1] &&
                        cz >= g.act_lo[2] && cz < g.act_hi[2];
    if (n_c && active) {
      unsigned long long S = 0;
      for (int seg = 0; seg < kMaxSeg; ++seg) {
        const Segment s = stencil_segment(g, cell_start, cx, cy, cz, seg);
        S += s.end - s.start;
      }
      const uint32_t tpi = targets_per_item(n_c, fine);
      const unsigned long long ntile = (n_c + tpi - 1) / tpi;
      const unsigned long long nchunk = (S + kSrcChunk - 1) / kSrcChunk;
      it = ntile * nchunk;
      w = (unsigned long long)n_c * S;
      wbig = n_c > 64u ? w : 0ull;
      const unsigned long long sp = (n_c <= kSplit8MaxCell || (fine && n_c <= kSplitMaxCell)) ? 7ull : (n_c <= kSplitMaxCell ? 3ull : 0ull);
      slots = ntile * tpi * ((S + sp) & ~sp);
      nmax = n_c;
    }
    items[c] = it;
  }
  // block reduction of the statistics
  for (int o = 16; o; o >>= 1) {
    w += __shfl_xor_sync(0xffffffffu, w, o);
    slots += __shfl_xor_sync(0xffffffffu, slots, o);
    wbig += __shfl_xor_sync(0xffffffffu, wbig, o);
    nmax = max(nmax, __shfl_xor_sync(0xffffffffu, nmax, o));
  }
  if ((threadIdx.x & 31) == 0) {
    if (w) atomicAdd(&flags->candidate_pairs, w);
    if (slots) atomicAdd(&flags->pair_slots, slots);
    if (wbig) atomicAdd(&flags->big_pairs, wbig);
    if (nmax) atomicMax(&flags->max_cell_count, nmax);
  }
}

// ------------------------------------------------------------------ 64-bit exclusive scan (3 kernels) --
constexpr int kScanThreads = 1024;
constexpr int kScanPerThread = 4;
constexpr int kScanBlock = kScanThreads * kScanPerThread;

__device__ __forceinline__ unsigned long long block_exclusive_scan(unsigned long long v, unsigned long long* total) {
  __shared__ unsigned long long wsum[32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  unsigned long long x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned long long y = __shfl_up_sync(0xffffffffu, x, o);
    if (lane >= o) x += y;
  }
  __syncthreads();  // protect wsum reuse across calls
  if (lane == 31) wsum[wid] = x;
  __syncthreads();
  if (wid == 0) {
    unsigned long long w = wsum[lane];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned long long y = __shfl_up_sync(0xffffffffu, w, o);
      if (lane >= o) w += y;
    }
    wsum[lane] = w;
  }
  __syncthreads();
  if (total) *total = wsum[31];
  return (wid ? wsum[wid - 1] : 0ull) + (x - v);
}

__global__ void __launch_bounds__(kScanThreads) k_scan_reduce(const unsigned long long* __restrict__ in, int n,
                                                               unsigned long long* __restrict__ block_sums) {
  const int base = blockIdx.x * kScanBlock + threadIdx.x * kScanPerThread;
  unsigned long long s = 0;
#pragma unroll
  for (int j = 0; j < kScanPerThread; ++j) s += (base + j < n) ? in[base + j] : 0ull;
  unsigned long long tot;
  block_exclusive_scan(s, &tot);
  if (threadIdx.x == 0) block_sums[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(kScanThreads) k_scan_top(unsigned long long* __restrict__ block_sums, int nb,
                                                            unsigned long long* __restrict__ total_out,
                                                            unsigned long long* __restrict__ total_out2) {
  const int base = threadIdx.x * kScanPerThread;
  unsigned long long v[kScanPerThread], s = 0;
#pragma unroll
  for (int j = 0; j < kScanPerThread; ++j) { v[j] = (base + j < nb) ? block_sums[base + j] : 0ull; s += v[j]; }
  unsigned long long tot;
  unsigned long long ex = block_exclusive_scan(s, &tot);
#pragma unroll
  for (int j = 0; j < kScanPerThread; ++j) { if (base + j < nb) block_sums[base + j] = ex; ex += v[j]; }
  if (threadIdx.x == 0) { *total_out = tot; *total_out2 = tot; }
}

__global__ void __launch_bounds__(kScanThreads) k_scan_apply(unsigned long long* __restrict__ data, int n,
                                                              const unsigned long long* __restrict__ block_sums) {
  const int base = blockIdx.x * kScanBlock + threadIdx.x * kScanPerThread;
  unsigned long long v[kScanPerThread], s = 0;
#pragma unroll
  for (int j = 0; j < kScanPerThread; ++j) { v[j] = (base + j < n) ? data[base + j] : 0ull; s += v[j]; }
  unsigned long long ex = block_exclusive_scan(s, nullptr) + block_sums[blockIdx.x];
#pragma unroll
  for (int j = 0; j < kScanPerThread; ++j) { if (base + j < n) data[base + j] = ex; ex += v[j]; }
}

// ------------------------------------------------------------------------------------ A5: PP force --
__device__ __forceinline__ float rsqrt_approx(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));   // one MUFU.RSQ
  return y;
}

__device__ __forceinline__ void red_add_f64(double* addr, double v) {
  asm volatile("red.global.add.f64 [%0], %1;" ::"l"(addr), "d"(v) : "memory");
}

struct __align__(16) WarpScratch {
  float4 src[kSrcTile];     // (x, y, z, m) of a staged source, relative to the item's reference point
  uint32_t seg_start[kMaxSeg + 1];   // stream offset of each segment; [kMaxSeg] = S
  uint32_t seg_base[kMaxSeg];        // sorted index of each segment's first particle
  float seg_ref[kMaxSeg][3];         // integer-valued reference point R_s of the segment's cells
  float seg_delta[kMaxSeg][3];       // R_s - R_t + periodic shift  (exact for integer box lengths)
};

// One work item for one warp.  TP = target pairs per lane (T = 2*TP targets per lane).
template <int TP, bool kUniformMass, int S>
__device__ __forceinline__ void process_item(WarpScratch& ws, const float4* __restrict__ sorted, const ForceConst& fc,
                                             uint32_t tgt_begin, uint32_t tgt_end, const float ref_t[3],
                                             uint32_t p0, uint32_t p1, double* __restrict__ acc64, int lane, float lane_zero) {
  // ---- targets: lane holds pairs (k, k+32) of each 64-block, negated and relative to R_t
  float2 ntx[TP], nty[TP], ntz[TP], ax[TP], ay[TP], az[TP];
#pragma unroll
  for (int t = 0; t < TP; ++t) {
    const uint32_t k0 = tgt_begin + t * (64 / S) + (lane & (32 / S - 1)), k1 = k0 + 32 / S;
    float4 a = make_float4(-fc.pad, -fc.pad, -fc.pad, 0.f), b = a;   // empty target slot: beyond rc of every source
    if (k0 < tgt_end) { a = __ldg(&sorted[k0]); a.x -= ref_t[0]; a.y -= ref_t[1]; a.z -= ref_t[2]; }
    if (k1 < tgt_end) { b = __ldg(&sorted[k1]); b.x -= ref_t[0]; b.y -= ref_t[1]; b.z -= ref_t[2]; }
    ntx[t] = make_float2(-a.x, -b.x);
    nty[t] = make_float2(-a.y, -b.y);
    ntz[t] = make_float2(-a.z, -b.z);
    ax[t] = ay[t] = az[t] = make_float2(0.f, 0.f);
  }
  const float2 e2 = make_float2(fc.eps2, fc.eps2);
  // c5*u + c4 needs two constants in one instruction, and an FFMA2 takes at most one uniform-register operand:
  // c4 is made a per-lane value on purpose (lane_zero is 0.0f, but not provably so), which keeps ptxas from also
  // demoting other constants to vector registers (a third vector operand costs the FMA pipe a third cycle).
  const float c4v = fc.nq[4] + lane_zero;
  const float2 c5 = make_float2(fc.nq[5], fc.nq[5]), c4 = make_float2(c4v, c4v);
  const float2 c3 = make_float2(fc.nq[3], fc.nq[3]), c2 = make_float2(fc.nq[2], fc.nq[2]);
  const float2 c1 = make_float2(fc.nq[1], fc.nq[1]), c0 = make_float2(fc.nq[0], fc.nq[0]);
  const float rc2e = fc.rc2e;

  int seg = 0;  // monotone per-lane segment cursor (stream positions only grow)
  for (uint32_t tile = p0; tile < p1; tile += kSrcTile) {
    // ---- stage up to kSrcTile stream positions into the warp-private tile
    __syncwarp();
#pragma unroll
    for (int j = 0; j < kSrcTile / 32; ++j) {
      const uint32_t p = tile + j * 32 + lane;
      float4 sv = make_float4(fc.pad, fc.pad, fc.pad, 0.f);   // empty source slot: cut off for every target (scale-independent)
      if (p < p1) {
        while (p >= ws.seg_start[seg + 1]) ++seg;
        const float4 v = __ldg(&sorted[ws.seg_base[seg] + (p - ws.seg_start[seg])]);
        const float x = (v.x - ws.seg_ref[seg][0]) + ws.seg_delta[seg][0];
        const float y = (v.y - ws.seg_ref[seg][1]) + ws.seg_delta[seg][1];
        const float z = (v.z - ws.seg_ref[seg][2]) + ws.seg_delta[seg][2];
        sv = make_float4(x, y, z, v.w);
      }
      ws.src[j * 32 + lane] = sv;
    }
    __syncwarp();
    // ---- pair loop: every source of the tile against the lane's 2*TP targets
    const int cnt = (int)min((uint32_t)kSrcTile, (p1 - tile + (uint32_t)(S - 1)) & ~(uint32_t)(S - 1));
    // Small-cell variants (S > 1) are unrolled to about 8 packed-pair bodies per trip: they run side by side on one SM
    // sub-partition (cells of 20..46 particles pick four of them), and bodies of 20 packed pairs each (7 KB of code per
    // variant) thrashed the instruction cache -- FMA-pipe utilisation fell from 83 % to 63 %.  The large-cell variant is
    // alone on the chip for most of its time: 8 sources x 4 packed pairs per trip gives ptxas the freedom to keep the
    // FMA pipe fed across the MUFU latencies (measured on config 3 at 128 registers: TP 2 / unroll 4 71.3 %, TP 3 /
    // unroll 4 72.7 %, TP 3 / unroll 16 73.9 %, TP 3 / unroll 32 73.5 %; at 168 registers: TP 4 / unroll 8 74.8 %,
    // TP 4 / unroll 12 74.3 %, TP 5 / unroll 8 72.3 % of FP32 peak).
#pragma unroll (S > 1 ? (TP >= 3 ? 2 : 4) : 8)
    for (int j = (S > 1 ? lane / (32 / S) : 0); j < cnt; j += S) {
      // one LDS.128 per source; the packed instructions broadcast the scalar to both halves (R.F32 operand form)
      const float4 sv = ws.src[j];
      const float2 sx = make_float2(sv.x, sv.x), sy = make_float2(sv.y, sv.y), sz = make_float2(sv.z, sv.z);
      const float2 sm = make_float2(sv.w, sv.w);
#pragma unroll
      for (int t = 0; t < TP; ++t) {
        const float2 dx = __fadd2_rn(sx, ntx[t]);
        const float2 dy = __fadd2_rn(sy, nty[t]);
        const float2 dz = __fadd2_rn(sz, ntz[t]);
        float2 u = __ffma2_rn(dx, dx, e2);
        u = __ffma2_rn(dy, dy, u);
        u = __ffma2_rn(dz, dz, u);
        const float2 r = make_float2(rsqrt_approx(u.x), rsqrt_approx(u.y));
        const float2 r2 = __fmul2_rn(r, r);
        float2 q = __ffma2_rn(c5, u, c4);
        q = __ffma2_rn(q, u, c3);
        q = __ffma2_rn(q, u, c2);
        q = __ffma2_rn(q, u, c1);
        q = __ffma2_rn(q, u, c0);
        float2 f = __ffma2_rn(r2, r, q);          // r^3 - Q(u)
        f.x = (u.x < rc2e) ? f.x : 0.f;           // strict cutoff (R5), plain truncation (R6)
        f.y = (u.y < rc2e) ? f.y : 0.f;
        if (!kUniformMass) f = __fmul2_rn(f, sm);
        ax[t] = __ffma2_rn(f, dx, ax[t]);
        ay[t] = __ffma2_rn(f, dy, ay[t]);
        az[t] = __ffma2_rn(f, dz, az[t]);
      }
    }
  }
  // ---- small-cell path: add the partial sums of the S source phases (lanes l, l + 32/S, ... hold the same targets)
  if (S > 1) {
#pragma unroll
    for (int t = 0; t < TP; ++t) {
#pragma unroll
      for (int o = 32 / S; o < 32; o <<= 1) {
        ax[t].x += __shfl_xor_sync(0xffffffffu, ax[t].x, o); ax[t].y += __shfl_xor_sync(0xffffffffu, ax[t].y, o);
        ay[t].x += __shfl_xor_sync(0xffffffffu, ay[t].x, o); ay[t].y += __shfl_xor_sync(0xffffffffu, ay[t].y, o);
        az[t].x += __shfl_xor_sync(0xffffffffu, az[t].x, o); az[t].y += __shfl_xor_sync(0xffffffffu, az[t].y, o);
      }
    }
    if (lane >= 32 / S) return;
  }
  // ---- fold the fp32 partial sums into the fp64 accumulators (sorted order)
#pragma unroll
  for (int t = 0; t < TP; ++t) {
    const uint32_t k0 = tgt_begin + t * (64 / S) + (lane & (32 / S - 1)), k1 = k0 + 32 / S;
    if (k0 < tgt_end) {
      red_add_f64(&acc64[3 * (size_t)k0 + 0], (double)ax[t].x);
      red_add_f64(&acc64[3 * (size_t)k0 + 1], (double)ay[t].x);
      red_add_f64(&acc64[3 * (size_t)k0 + 2], (double)az[t].x);
    }
    if (k1 < tgt_end) {
      red_add_f64(&acc64[3 * (size_t)k1 + 0], (double)ax[t].y);
      red_add_f64(&acc64[3 * (size_t)k1 + 1], (double)ay[t].y);
      red_add_f64(&acc64[3 * (size_t)k1 + 2], (double)az[t].y);
    }
  }
}

template <bool kUniformMass, int kBuild>
__global__ void __launch_bounds__(PPBuild<kBuild>::kThreads, PPBuild<kBuild>::kCtasPerSm)
k_pp_force(const float4* __restrict__ sorted, const uint32_t* __restrict__ cell_start,
           const unsigned long long* __restrict__ item_prefix, Geometry g, ForceConst fc, DevFlags* flags,
           double* __restrict__ acc64) {
  // the build is a device-side fact (found by the plan kernel): both are launched, one returns at once
  if ((2ull * flags->big_pairs > flags->candidate_pairs ? 1 : 0) != kBuild) return;
  __shared__ WarpScratch scratch[PPBuild<kBuild>::kThreads / 32];
  const int lane = threadIdx.x & 31;
  WarpScratch& ws = scratch[threadIdx.x >> 5];
  const unsigned long long total = flags->total_items;
  const float lane_zero = __uint_as_float(__ldg(&flags->pad0 + (lane >> 5)));   // 0.0f (pad0 is cleared by every mesh build)

  for (;;) {
    unsigned long long idx = 0;
    if (lane == 0) idx = atomicAdd(&flags->item_counter, 1ull);
    idx = __shfl_sync(0xffffffffu, idx, 0);
    if (idx >= total) break;

    // ---- 32-ary search: largest c with item_prefix[c] <= idx  (item_prefix[ncells] = total > idx)
    int lo = 0, hi = g.ncells;            // invariant: prefix[lo] <= idx < prefix[hi]
    while (hi - lo > 1) {
      const int step = (hi - lo + 31) / 32;
      const int probe = lo + lane * step;
      const bool le = (probe < hi) && (__ldg(&item_prefix[probe]) <= idx);
      const uint32_t ballot = __ballot_sync(0xffffffffu, le);
      const int k = __popc(ballot);       // >= 1 (probe == lo always qualifies); qualifying lanes form a prefix
      const int nlo = lo + (k - 1) * step;
      hi = min(hi, nlo + step);
      lo = nlo;
    }
    const int c = lo;
    const unsigned long long local = idx - __ldg(&item_prefix[c]);   // 64-bit: one cell can hold > 2^32 items
    const uint32_t cs0 = __ldg(&cell_start[c]), cs1 = __ldg(&cell_start[c + 1]);
    const uint32_t n_c = cs1 - cs0;
    const uint32_t tpi = targets_per_item(n_c, fc.fine_items);
    const uint32_t ntile = (n_c + tpi - 1) / tpi;
    const uint32_t tile = (uint32_t)(local % ntile);              // chunk-major: neighbours share sources
    const unsigned long long chunk = local / ntile;
    const int cx = c % g.ncell[0], cy = (c / g.ncell[0]) % g.ncell[1], cz = c / (g.ncell[0] * g.ncell[1]);

    // ---- segment table of this cell's source stream (lanes 0..17), prefix by warp scan
    float ref_t[3] = {floorf(cx * g.cell_w[0]), floorf(cy * g.cell_w[1]), floorf(cz * g.cell_w[2])};
    uint32_t len = 0;
    Segment s;
    if (lane < kMaxSeg) {
      s = stencil_segment(g, cell_start, cx, cy, cz, lane);
      len = s.end - s.start;
    }
    uint32_t incl = len;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t y = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += y;
    }
    __syncwarp();
    if (lane < kMaxSeg) {
      ws.seg_start[lane] = incl - len;
      ws.seg_base[lane] = s.start;
      const float rs[3] = {floorf(s.xlo * g.cell_w[0]), floorf(s.cy * g.cell_w[1]), floorf(s.cz * g.cell_w[2])};
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        ws.seg_ref[lane][a] = rs[a];
        ws.seg_delta[lane][a] = (float)(((double)rs[a] - (double)ref_t[a]) + (double)s.shift[a]);
      }
    }
    const uint32_t S = __shfl_sync(0xffffffffu, incl, kMaxSeg - 1);
    if (lane == 0) ws.seg_start[kMaxSeg] = S;
    __syncwarp();

    const uint32_t p0 = (uint32_t)min(chunk * (unsigned long long)kSrcChunk, (unsigned long long)S), p1 = min(S, p0 + kSrcChunk);
    const uint32_t tb = cs0 + tile * tpi, te = min(cs1, tb + tpi);
    if (n_c <= 8u)
      process_item<1, kUniformMass, 8>(ws, sorted, fc, tb, te, ref_t, p0, p1, acc64, lane, lane_zero);
    else if (n_c <= 16u || (fc.fine_items && n_c <= kSplitMaxCell))
      process_item<2, kUniformMass, 8>(ws, sorted, fc, tb, te, ref_t, p0, p1, acc64, lane, lane_zero);
    else if (n_c <= 24u)
      process_item<3, kUniformMass, 8>(ws, sorted, fc, tb, te, ref_t, p0, p1, acc64, lane, lane_zero);
    else if (n_c <= 32u)
      process_item<4, kUniformMass, 8>(ws, sorted, fc, tb, te, ref_t, p0, p1, acc64, lane, lane_zero);
    else if (n_c <= kSplit8MaxCell)
      process_item<5, kUniformMass, 8>(ws, sorted, fc, tb, te, ref_t, p0, p1, acc64, lane, lane_zero);
    else if (n_c <= kSplitMaxCell)
      process_item<3, kUniformMass, 4>(ws, sorted, fc, tb, te, ref_t, p0, p1, acc64, lane, lane_zero);
    else if (n_c <= 64u)
      process_item<1, kUniformMass, 1>(ws, sorted, fc, tb, te, ref_t, p0, p1, acc64, lane, lane_zero);
    else
      process_item<kBigTP, kUniformMass, 1>(ws, sorted, fc, tb, te, ref_t, p0, p1, acc64, lane, lane_zero);
  }
}

// --------------------------------------------------------------------------------- A6: write-back --
// Direct form (small n: the whole acc / vel arrays sit in L2): acc[perm[k]] = (float)(acc64[k] * scale), and with kKick
// the sub-cycled kick of A7 on the same particle, v <- fmaf(a, kdt, v) (bit-identical to k_kick on the written acc).
template <bool kKick>
__global__ void __launch_bounds__(256) k_write_back(const double* __restrict__ acc64, const uint32_t* __restrict__ perm,
                                                     int64_t n, float scale, float4* __restrict__ acc,
                                                     float4* __restrict__ vel, float kdt) {
  // 4 independent elements per thread and trip: the scattered 16-byte stores are the slow part, keep many in flight
  constexpr int U = 4;
  const double s = (double)scale;
  for (int64_t k0 = (int64_t)blockIdx.x * blockDim.x * U + threadIdx.x; k0 < n; k0 += (int64_t)gridDim.x * blockDim.x * U) {
    double a[U][3];
    uint32_t dst[U];
    float4 v[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t k = k0 + (int64_t)u * blockDim.x;
      if (k < n) {
        dst[u] = __ldcs(&perm[k]);
        a[u][0] = __ldcs(&acc64[3 * k + 0]); a[u][1] = __ldcs(&acc64[3 * k + 1]); a[u][2] = __ldcs(&acc64[3 * k + 2]);
        if (kKick) v[u] = vel[dst[u]];
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t k = k0 + (int64_t)u * blockDim.x;
      if (k < n) {
        const float4 o = make_float4((float)(a[u][0] * s), (float)(a[u][1] * s), (float)(a[u][2] * s), 0.f);
        acc[dst[u]] = o;
        if (kKick) {
          v[u].x = __fmaf_rn(o.x, kdt, v[u].x); v[u].y = __fmaf_rn(o.y, kdt, v[u].y); v[u].z = __fmaf_rn(o.z, kdt, v[u].z);
          vel[dst[u]] = v[u];
        }
      }
    }
  }
}

// Bucketed form (n >= kUnsortMinN).  perm is a random permutation of the caller's order in the worst case,
// so the direct scatter touches one 32-byte DRAM sector per 16-byte store with no locality (measured: 1.43 ms for 2^25
// particles, 0.145 of the HBM copy rate; a scatter into L2-sized windows is no better -- every 16-byte store to a
// sector that is not resident costs a DRAM fill and the sector is written back twice).  Instead the elements
// (ax, ay, az, destination index in the .w lane) are radix-partitioned by DESTINATION, most significant digit first,
// in two (n <= 2^28) or three coalesced passes down to windows of 4096 consecutive destinations:
//   k_unsort_partition  tiles of 4096 elements; bucket = destination >> shift.  perm is a permutation, so bucket b
//                       holds exactly the destinations [b << shift, (b + 1) << shift): its place in the output is known
//                       without a histogram and one global atomic per tile and bucket reserves the tile's run in it.
//                       Unordered inside a bucket (ranks from shared-memory atomics): the order does not matter.
//   k_unsort_final      one CTA per window: the 4096 elements are placed at (destination & 4095) in shared memory and
//                       leave as a linear stream -- with the kick of A7 fused in, vel is read and written linearly too.
constexpr int kUnsortThreads = 512;
constexpr int kUnsortTile = 4096;
constexpr int kUnsortWinBits = 12;                        // final windows: 4096 destinations = one shared-memory tile
constexpr int kUnsortItems = kUnsortTile / kUnsortThreads;
constexpr int kUnsortMaxBins = 256;

// kSrc 0: first level, elements made from the fp64 accumulators (x scale) and perm; 1: first level, elements made from
// the xyz of a sorted float4 array and perm (the sub-cycle's positions / velocities going back to the caller's order);
// 2: a later level, reads the previous level's elements.
// prev_shift: the input is already grouped in windows of 2^prev_shift destinations (31: the whole array).
template <int kSrc>
__global__ void __launch_bounds__(kUnsortThreads, 2) k_unsort_partition(
    const double* __restrict__ acc64, const uint32_t* __restrict__ perm, const float4* __restrict__ in, int64_t n,
    float scale, int prev_shift, int shift, uint32_t* __restrict__ cursor /*[n >> shift, +1], cleared*/,
    float4* __restrict__ out) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float4* stile = (float4*)smem_raw;                       // [kUnsortTile] bucket order
  uint32_t* cnt = (uint32_t*)(stile + kUnsortTile);        // [kUnsortMaxBins]
  uint32_t* tstart = cnt + kUnsortMaxBins;                 // start of the bucket inside the tile
  uint32_t* gbase = tstart + kUnsortMaxBins;               // start of the tile's run inside the bucket
  uint32_t* wsum = gbase + kUnsortMaxBins;                 // [32]
  const double s = (double)scale;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const uint32_t lmask = (1u << (prev_shift - shift)) - 1u;      // buckets per input window (<= kUnsortMaxBins)
  const int64_t ntiles = (n + kUnsortTile - 1) / kUnsortTile;
  for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
    const int64_t base = t * kUnsortTile;
    const int tile_n = (int)min((int64_t)kUnsortTile, n - base);
    const uint32_t bucket0 = (uint32_t)(base >> prev_shift) << (prev_shift - shift);   // first bucket of the tile's window
    if ((int)threadIdx.x < kUnsortMaxBins) cnt[threadIdx.x] = 0u;
    __syncthreads();
    float4 v[kUnsortItems];
    uint32_t rk[kUnsortItems];
#pragma unroll
    for (int u = 0; u < kUnsortItems; ++u) {
      const int e = u * kUnsortThreads + threadIdx.x;
      v[u] = make_float4(0.f, 0.f, 0.f, 0.f);
      if (e < tile_n) {
        const int64_t k = base + e;
        if (kSrc == 0) {
          const uint32_t dst = __ldcs(&perm[k]);
          v[u] = make_float4((float)(__ldcs(&acc64[3 * k + 0]) * s), (float)(__ldcs(&acc64[3 * k + 1]) * s),
                             (float)(__ldcs(&acc64[3 * k + 2]) * s), __uint_as_float(dst));
        } else {
          v[u] = __ldcs(&in[k]);
          if (kSrc == 1) v[u].w = __uint_as_float(__ldcs(&perm[k]));
        }
      }
    }
#pragma unroll
    for (int u = 0; u < kUnsortItems; ++u)
      if (u * kUnsortThreads + (int)threadIdx.x < tile_n) rk[u] = atomicAdd(&cnt[(__float_as_uint(v[u].w) >> shift) & lmask], 1u);
    __syncthreads();
    // bucket threads: reserve the tile's run in every bucket, exclusive scan of the counts over the buckets
    if ((int)threadIdx.x < kUnsortMaxBins) {
      const uint32_t c = cnt[threadIdx.x];
      gbase[threadIdx.x] = c ? atomicAdd(&cursor[bucket0 + threadIdx.x], c) : 0u;
      uint32_t x = c;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
      if (lane == 31) wsum[w] = x;
      asm volatile("bar.sync 1, %0;" ::"n"(kUnsortMaxBins) : "memory");
      uint32_t off = 0;
      for (int r = 0; r < w; ++r) off += wsum[r];
      tstart[threadIdx.x] = off + x - c;
    }
    __syncthreads();
#pragma unroll
    for (int u = 0; u < kUnsortItems; ++u)
      if (u * kUnsortThreads + (int)threadIdx.x < tile_n) stile[tstart[(__float_as_uint(v[u].w) >> shift) & lmask] + rk[u]] = v[u];
    __syncthreads();
#pragma unroll
    for (int u = 0; u < kUnsortItems; ++u) {
      const int q = u * kUnsortThreads + threadIdx.x;
      if (q < tile_n) {
        const float4 e = stile[q];
        const uint32_t b = __float_as_uint(e.w) >> shift, bl = b & lmask;
        out[((size_t)b << shift) + gbase[bl] + ((uint32_t)q - tstart[bl])] = e;
      }
    }
    __syncthreads();
  }
}

// kMode 0: acc = (x, y, z, 0); 1: the same and the kick v <- fmaf(a, kdt, v) on vel; 2: xyz written into acc's elements,
// their .w lanes kept (positions with their masses, velocities).
template <int kMode>
__global__ void __launch_bounds__(kUnsortThreads, 2) k_unsort_final(const float4* __restrict__ buf, int64_t n,
                                                                     float4* __restrict__ acc, float4* __restrict__ vel,
                                                                     float kdt) {
  constexpr bool kKick = kMode == 1;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float4* stile = (float4*)smem_raw;                       // [kUnsortTile] destination order
  const int64_t nwin = (n + kUnsortTile - 1) / kUnsortTile;
  for (int64_t t = blockIdx.x; t < nwin; t += gridDim.x) {
    const int64_t base = t * kUnsortTile;
    const int win_n = (int)min((int64_t)kUnsortTile, n - base);
    {
      float4 e[kUnsortItems];
#pragma unroll
      for (int u = 0; u < kUnsortItems; ++u) {
        const int q = u * kUnsortThreads + threadIdx.x;
        if (q < win_n) e[u] = __ldcs(&buf[base + q]);
      }
#pragma unroll
      for (int u = 0; u < kUnsortItems; ++u)
        if (u * kUnsortThreads + (int)threadIdx.x < win_n) stile[__float_as_uint(e[u].w) & (kUnsortTile - 1)] = e[u];
    }
    __syncthreads();
    // linear output, four elements per thread in flight (with the kick: their velocities too)
#pragma unroll 1
    for (int h = 0; h < kUnsortItems; h += 4) {
      float4 v[4];
      if (kMode != 0) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int q = (h + u) * kUnsortThreads + threadIdx.x;
          if (q < win_n) v[u] = kKick ? vel[base + q] : acc[base + q];
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int q = (h + u) * kUnsortThreads + threadIdx.x;
        if (q < win_n) {
          const float4 a = stile[q];
          acc[base + q] = make_float4(a.x, a.y, a.z, kMode == 2 ? v[u].w : 0.f);
          if (kKick) {
            v[u].x = __fmaf_rn(a.x, kdt, v[u].x); v[u].y = __fmaf_rn(a.y, kdt, v[u].y); v[u].z = __fmaf_rn(a.z, kdt, v[u].z);
            vel[base + q] = v[u];
          }
        }
      }
    }
    __syncthreads();
  }
}

// ----------------------------------------------------------------------------- A7: kick, and stream --
__global__ void __launch_bounds__(256) k_kick(float4* __restrict__ vel, const float4* __restrict__ acc, float kdt, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    float4 v = vel[i];
    const float4 a = __ldg(&acc[i]);
    v.x = __fmaf_rn(a.x, kdt, v.x);
    v.y = __fmaf_rn(a.y, kdt, v.y);
    v.z = __fmaf_rn(a.z, kdt, v.z);
    vel[i] = v;
  }
}

__global__ void __launch_bounds__(256) k_stream(float4* __restrict__ pos, const float4* __restrict__ vel, float dt,
                                                 float Lx, float Ly, float Lz, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    float4 p = pos[i];
    const float4 v = __ldg(&vel[i]);
    p.x = wrap_coord(__fmaf_rn(v.x, dt, p.x), Lx);
    p.y = wrap_coord(__fmaf_rn(v.y, dt, p.y), Ly);
    p.z = wrap_coord(__fmaf_rn(v.z, dt, p.z), Lz);
    pos[i] = p;
  }
}

// ------------------------------------------------------------------------------------ host launchers --
void query_force_occupancy(int* blocks_per_sm /*[2]*/) {
  int a = 0, b = 0;
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&a, k_pp_force<true, 0>, PPBuild<0>::kThreads, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, k_pp_force<false, 0>, PPBuild<0>::kThreads, 0);
  blocks_per_sm[0] = a < b ? a : b;
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&a, k_pp_force<true, 1>, PPBuild<1>::kThreads, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, k_pp_force<false, 1>, PPBuild<1>::kThreads, 0);
  blocks_per_sm[1] = a < b ? a : b;
  for (int k = 0; k < 2; ++k)
    if (blocks_per_sm[k] < 1) blocks_per_sm[k] = 1;
}

cudaError_t launch_scan_u64(cudaStream_t st, unsigned long long* data, int n, unsigned long long* tmp,
                            unsigned long long* total_out, unsigned long long* total_out2) {
  const int nb = (n + kScanBlock - 1) / kScanBlock;     // <= 4096 blocks (n <= 2^24): one top-level block scans them
  k_scan_reduce<<<nb, kScanThreads, 0, st>>>(data, n, tmp);
  k_scan_top<<<1, kScanThreads, 0, st>>>(tmp, nb, total_out, total_out2);
  k_scan_apply<<<nb, kScanThreads, 0, st>>>(data, n, tmp);
  return cudaGetLastError();
}

cudaError_t launch_accel_sorted(srpp_ctx* c) {
  cudaStream_t st = c->stream;
  const int64_t n = c->n;
  const int32_t ncells = c->geo.ncells;
  cudaError_t e;
  if (n == 0) return cudaSuccess;
  // reset queue head + statistics (keep the binning flags)
  if ((e = cudaMemsetAsync(&c->flags->max_cell_count, 0, sizeof(DevFlags) - offsetof(DevFlags, max_cell_count), st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(c->acc64, 0, sizeof(double) * 3 * (size_t)n, st)) != cudaSuccess) return e;
  // fewer than 64 particles per resident warp (of build 0, the one tiny problems take): finer items
  c->fc.fine_items = n < (int64_t)c->num_sms * c->force_blocks_per_sm[0] * (PPBuild<0>::kThreads / 32) * 64 ? 1 : 0;
  k_plan_items<<<(ncells + 255) / 256, 256, 0, st>>>(c->cell_start, c->geo, c->fc.fine_items, c->item_prefix, c->flags);
  if ((e = launch_scan_u64(st, c->item_prefix, ncells, c->scan_tmp, &c->flags->total_items, &c->item_prefix[ncells])) != cudaSuccess) return e;
  const int grid0 = c->num_sms * c->force_blocks_per_sm[0], grid1 = c->num_sms * c->force_blocks_per_sm[1];
  if (c->timing) cudaEventRecord(c->ev[kEvForce0], st);
  if (c->uniform_mass) {
    k_pp_force<true, 0><<<grid0, PPBuild<0>::kThreads, 0, st>>>(c->sorted, c->cell_start, c->item_prefix, c->geo, c->fc, c->flags, c->acc64);
    k_pp_force<true, 1><<<grid1, PPBuild<1>::kThreads, 0, st>>>(c->sorted, c->cell_start, c->item_prefix, c->geo, c->fc, c->flags, c->acc64);
  } else {
    k_pp_force<false, 0><<<grid0, PPBuild<0>::kThreads, 0, st>>>(c->sorted, c->cell_start, c->item_prefix, c->geo, c->fc, c->flags, c->acc64);
    k_pp_force<false, 1><<<grid1, PPBuild<1>::kThreads, 0, st>>>(c->sorted, c->cell_start, c->item_prefix, c->geo, c->fc, c->flags, c->acc64);
  }
  if (c->timing) cudaEventRecord(c->ev[kEvForce1], st);
  c->launches += 6;
  return cudaGetLastError();
}

// Bucketed un-sort of one array (n >= kUnsortMinN): `sorted_src` == nullptr takes the fp64 accumulators (A6), else
// the xyz of a sorted float4 array; mode as in k_unsort_final.
static cudaError_t launch_unsort(srpp_ctx* c, const float4* sorted_src, float scale, int mode, float4* dst, float4* vel, float kdt) {
  const int64_t n = c->n;
  cudaStream_t st = c->stream;
  // levels: the window index (destination >> 12) has `tb` bits, split evenly over the levels, <= 8 bits each
  const int64_t nwin = (n + kUnsortTile - 1) >> kUnsortWinBits;
  int tb = 1;
  while (((int64_t)1 << tb) < nwin) ++tb;
  const int nlev = (tb + 7) / 8;
  const int o = c->sorted == c->sorted_buf[0] ? 1 : 0;            // the idle partners of the sub-cycle's ping-pong buffers
  float4* bufs[2] = {c->sorted_buf[o], c->vel_s[o]};
  const size_t smem = (size_t)kUnsortTile * sizeof(float4) + (3 * kUnsortMaxBins + 32) * sizeof(uint32_t);
  const size_t smem_fin = (size_t)kUnsortTile * sizeof(float4);
  cudaError_t e;
  if (!c->unsort_attr_set) {
    if ((e = cudaFuncSetAttribute(k_unsort_partition<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_unsort_partition<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_unsort_partition<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_unsort_final<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_fin)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_unsort_final<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_fin)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_unsort_final<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_fin)) != cudaSuccess) return e;
    c->unsort_attr_set = true;
  }
  if ((e = cudaMemsetAsync(c->unsort_cursor, 0, unsort_cursor_bytes(n), st)) != cudaSuccess) return e;
  const int64_t ntiles = (n + kUnsortTile - 1) / kUnsortTile;
  const int grid = (int)std::min<int64_t>(ntiles, (int64_t)c->num_sms * 2);
  int prev_shift = 31, bits_left = tb;
  uint32_t* cursor = c->unsort_cursor;
  const float4* in = nullptr;
  for (int l = 0; l < nlev; ++l) {
    const int bl = (bits_left + (nlev - l) - 1) / (nlev - l);      // bits of this level
    bits_left -= bl;
    const int shift = kUnsortWinBits + bits_left;
    float4* out = bufs[l & 1];
    if (l == 0 && !sorted_src) k_unsort_partition<0><<<grid, kUnsortThreads, smem, st>>>(c->acc64, c->perm, nullptr, n, scale, prev_shift, shift, cursor, out);
    else if (l == 0) k_unsort_partition<1><<<grid, kUnsortThreads, smem, st>>>(nullptr, c->perm, sorted_src, n, 1.f, prev_shift, shift, cursor, out);
    else k_unsort_partition<2><<<grid, kUnsortThreads, smem, st>>>(nullptr, nullptr, in, n, 1.f, prev_shift, shift, cursor, out);
    cursor += ((n - 1) >> shift) + 1;                               // this level's buckets
    prev_shift = shift;
    in = out;
  }
  if (mode == 1) k_unsort_final<1><<<grid, kUnsortThreads, smem_fin, st>>>(in, n, dst, vel, kdt);
  else if (mode == 2) k_unsort_final<2><<<grid, kUnsortThreads, smem_fin, st>>>(in, n, dst, nullptr, 0.f);
  else k_unsort_final<0><<<grid, kUnsortThreads, smem_fin, st>>>(in, n, dst, nullptr, 0.f);
  c->launches += (uint64_t)nlev + 1;
  return cudaGetLastError();
}

cudaError_t launch_write_back(srpp_ctx* c, float4* acc, float4* vel, float kdt) {
  const int64_t n = c->n;
  if (n == 0) return cudaSuccess;
  cudaStream_t st = c->stream;
  const float scale = c->uniform_mass ? c->mass0 : 1.0f;
  if (n < kUnsortMinN) {
    const int grid_wb = (int)std::min<int64_t>((n + 1023) / 1024, (int64_t)c->num_sms * 16);
    if (vel) k_write_back<true><<<grid_wb, 256, 0, st>>>(c->acc64, c->perm, n, scale, acc, vel, kdt);
    else k_write_back<false><<<grid_wb, 256, 0, st>>>(c->acc64, c->perm, n, scale, acc, nullptr, 0.f);
    c->launches += 1;
    return cudaGetLastError();
  }
  return launch_unsort(c, nullptr, scale, vel ? 1 : 0, acc, vel, kdt);
}

// xyz of a sorted array back into the caller's array (its .w lanes are kept); n >= kUnsortMinN only
cudaError_t launch_unsort_xyz(srpp_ctx* c, const float4* sorted_src, float4* dst) {
  return launch_unsort(c, sorted_src, 1.f, 2, dst, nullptr, 0.f);
}

cudaError_t launch_accel(srpp_ctx* c, float4* acc, float4* vel, float kdt) {
  cudaStream_t st = c->stream;
  if (c->n == 0) return cudaSuccess;
  if (c->timing) cudaEventRecord(c->ev[kEvAccel0], st);
  cudaError_t e = launch_accel_sorted(c);
  if (e == cudaSuccess) e = launch_write_back(c, acc, vel, kdt);
  if (c->timing) { cudaEventRecord(c->ev[kEvAccel1], st); c->ev_accel_valid = true; }
  return e;
}

cudaError_t launch_kick(srpp_ctx* c, float4* vel, const float4* acc, float kdt, int64_t n) {
  if (n == 0) return cudaSuccess;
  const int grid_ew = (int)std::min<int64_t>((n + 255) / 256, (int64_t)c->num_sms * 16);
  k_kick<<<grid_ew, 256, 0, c->stream>>>(vel, acc, kdt, n);
  c->launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_stream(srpp_ctx* c, float4* pos_mass, const float4* vel, float dt, int64_t n) {
  if (n == 0) return cudaSuccess;
  const int grid_ew = (int)std::min<int64_t>((n + 255) / 256, (int64_t)c->num_sms * 16);
  k_stream<<<grid_ew, 256, 0, c->stream>>>(pos_mass, vel, dt, c->params.box[0], c->params.box[1], c->params.box[2], n);
  c->launches += 1;
  return cudaGetLastError();
}

}  // namespace srpp
