// srpp_subcycle.cu -- the short-range sub-cycle in SORTED space with an incremental re-bin (
// PAPER.md:73 "short-range force timestep": evolve, update the active particles, stream the passive ones).
//
//   nsub x {  x <- stream(x, v, dt/2);  a = accel(x);  v <- kick(v, a, kdt);  x <- stream(x, v, dt/2)  }       (reading R20)
//
// Between the first and the last sub-step nothing leaves chaining-mesh order: positions, velocities and the permutation
// stay sorted by (cell, original index), the kick and both half streams are one coalesced kernel (k_kick_stream) that
// reads the fp64 accumulators of the force kernel directly (the scattered write-back A6 and the re-read of acc by a
// separate kick disappear), and the mesh is repaired instead of rebuilt:
//   * k_kick_stream also computes the new cell of every particle; a particle whose cell changed is a MOVER.  Movers mark
//     their original index in a bit mask and append their slot to an (unordered) list.
//   * The movers are ranked by original index through the bit mask (prefix of popcounts), gathered in that order, and
//     sorted by new cell with the SAME stable counting sort as a full build -> (new cell, original index) order.
//   * Stayers keep their relative order.  With F = exclusive prefix of the mover flags over the old slots, Mstart = the
//     movers' cell_start and CS = the old cell_start:
//         stayer at old slot k, cell c:   new slot = k - F[k] + lower_bound(movers of c by original index, index of k)
//         mover r (cell c, index i):      new slot = p - F[p] + r,   p = lower_bound(old slots of c by original index, i)
//         cell_start'[c] = CS[c] - F[CS[c]] + Mstart[c]
//     (F is kept as one flag bit per slot + a prefix per 32-slot word; cell ids are recomputed from the positions)
//     which is exactly the merge of two sequences sorted by (cell, original index): the result is bit-identical to the
//     oracle's stable counting sort of the new positions (tested after every sub-step).
//   * More movers than the second buffer set holds (n/4), or n > 2^29: the state is scattered back to the caller's
//     order and the mesh is rebuilt in full.
#include <math.h>
#include <stdio.h>

#include <algorithm>

#include "srpp_internal.cuh"

namespace srpp {

constexpr int kSubTile = 1024;          // sorted slots per CTA of the slot-wise kernels
constexpr int kSubThreads = 256;

struct SubCounters {                    // device block (cleared before every k_kick_stream)
  unsigned long long movers;
  unsigned long long pad[3];
};

__global__ void __launch_bounds__(256) k_gather_f4(const float4* __restrict__ src, const uint32_t* __restrict__ perm, int64_t n,
                                                    float4* __restrict__ dst) {
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x)
    dst[k] = __ldg(&src[__ldg(&perm[k])]);
}

__global__ void __launch_bounds__(256) k_scatter2_f4(const float4* __restrict__ a_sorted, const float4* __restrict__ b_sorted,
                                                      const uint32_t* __restrict__ perm, int64_t n, float4* __restrict__ a,
                                                      float4* __restrict__ b) {
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
    const uint32_t i = __ldg(&perm[k]);
    a[i] = a_sorted[k];
    b[i] = b_sorted[k];
  }
}

// kick + half stream (+ the next sub-step's first half stream) in sorted space; mover detection.
// Arithmetic identical to k_write_back + k_kick + k_stream: a = (float)(acc64 * scale), v = fmaf(a, kdt, v),
// x = wrap(fmaf(v, half, x)) once or twice.  A CTA owns 1024 consecutive slots; a warp's 32 lanes own 32 consecutive
// slots per trip, so the ballot of the mover predicate IS the flag word of those slots (no atomics).  The movers' slots
// are collected in shared memory and appended to the global list with ONE atomic per CTA (a per-warp atomic on the one
// counter serialised the whole pass: 1.5 ms instead of 0.5 ms at 2^25 particles).
__global__ void __launch_bounds__(kSubThreads) k_kick_stream(
    float4* __restrict__ pos, float4* __restrict__ vel, const double* __restrict__ acc64, const uint32_t* __restrict__ perm,
    int64_t n, Geometry g, float scale, float kdt, float half, int twice, uint32_t* __restrict__ flag_words,
    uint32_t* __restrict__ mover_mask, uint32_t* __restrict__ mover_slots, int64_t m_cap,
    unsigned long long* __restrict__ tile_movers, SubCounters* __restrict__ ctr) {
  __shared__ uint32_t s_list[kSubTile];
  __shared__ uint32_t s_count;
  __shared__ unsigned long long s_base;
  if (threadIdx.x == 0) s_count = 0u;
  __syncthreads();
  const int64_t base = (int64_t)blockIdx.x * kSubTile;
  const double s = (double)scale;
  const int lane = threadIdx.x & 31;
#pragma unroll
  for (int u = 0; u < kSubTile / kSubThreads; ++u) {
    const int64_t k = base + threadIdx.x + u * kSubThreads;
    bool mover = false;
    if (k < n) {
      float4 x = pos[k], v = vel[k];
      const uint32_t ko = cell_key(x, g);
      const float ax = (float)(acc64[3 * k + 0] * s), ay = (float)(acc64[3 * k + 1] * s), az = (float)(acc64[3 * k + 2] * s);
      v.x = __fmaf_rn(ax, kdt, v.x); v.y = __fmaf_rn(ay, kdt, v.y); v.z = __fmaf_rn(az, kdt, v.z);
      x.x = wrap_coord(__fmaf_rn(v.x, half, x.x), g.box[0]);
      x.y = wrap_coord(__fmaf_rn(v.y, half, x.y), g.box[1]);
      x.z = wrap_coord(__fmaf_rn(v.z, half, x.z), g.box[2]);
      if (twice) {
        x.x = wrap_coord(__fmaf_rn(v.x, half, x.x), g.box[0]);
        x.y = wrap_coord(__fmaf_rn(v.y, half, x.y), g.box[1]);
        x.z = wrap_coord(__fmaf_rn(v.z, half, x.z), g.box[2]);
      }
      pos[k] = x; vel[k] = v;
      mover = cell_key(x, g) != ko;
    }
    const uint32_t bal = __ballot_sync(0xffffffffu, mover);
    if (lane == 0 && base + (threadIdx.x & ~31) + u * kSubThreads < n) flag_words[(base + (threadIdx.x & ~31) + u * kSubThreads) >> 5] = bal;
    if (bal) {
      uint32_t at = 0;
      if (lane == 0) at = atomicAdd(&s_count, (uint32_t)__popc(bal));
      at = __shfl_sync(0xffffffffu, at, 0);
      if (mover) {
        const uint32_t i = __ldg(&perm[k]);
        atomicOr(&mover_mask[i >> 5], 1u << (i & 31));
        s_list[at + __popc(bal & ((1u << lane) - 1u))] = (uint32_t)k;
      }
    }
  }
  __syncthreads();
  const uint32_t cnt = s_count;
  if (threadIdx.x == 0) {
    tile_movers[blockIdx.x] = (unsigned long long)cnt;
    s_base = cnt ? atomicAdd(&ctr->movers, (unsigned long long)cnt) : 0ull;
  }
  __syncthreads();
  const unsigned long long gb = s_base;
  for (uint32_t q = threadIdx.x; q < cnt; q += kSubThreads)
    if ((int64_t)(gb + q) < m_cap) mover_slots[gb + q] = s_list[q];
}

// word_prefix[j] = movers in the slots before flag word j (tile_prefix = exclusive scan of the per-tile counts)
__global__ void __launch_bounds__(256) k_word_prefix(const uint32_t* __restrict__ flag_words, int64_t nwords_slots,
                                                      const unsigned long long* __restrict__ tile_prefix,
                                                      uint32_t* __restrict__ word_prefix) {
  const int64_t tile = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);        // one warp per tile of 32 words
  const int lane = threadIdx.x & 31;
  const int64_t j = tile * 32 + lane;
  if (tile * 32 >= nwords_slots) return;
  const uint32_t c = j < nwords_slots ? (uint32_t)__popc(flag_words[j]) : 0u;
  uint32_t x = c;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
  if (j < nwords_slots) word_prefix[j] = (uint32_t)tile_prefix[tile] + x - c;
}

// F(p) = movers among the old slots < p
__device__ __forceinline__ uint32_t movers_before(const uint32_t* __restrict__ flag_words, const uint32_t* __restrict__ word_prefix,
                                                  uint32_t p, uint32_t n, uint32_t m) {
  if (p >= n) return m;
  return __ldg(&word_prefix[p >> 5]) + (uint32_t)__popc(__ldg(&flag_words[p >> 5]) & ((1u << (p & 31)) - 1u));
}

__global__ void __launch_bounds__(256) k_popc_words(const uint32_t* __restrict__ mask, int64_t nw, unsigned long long* __restrict__ out) {
  const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (w < nw) out[w] = (unsigned long long)__popc(mask[w]);
}

// the j-th mover in ascending original index: its slot and its (new) position
__global__ void __launch_bounds__(256) k_mover_place(const uint32_t* __restrict__ mover_slots, int64_t m,
                                                      const uint32_t* __restrict__ perm, const uint32_t* __restrict__ mask,
                                                      const unsigned long long* __restrict__ wprefix,
                                                      const float4* __restrict__ pos, uint32_t* __restrict__ slot_by_rank,
                                                      float4* __restrict__ mover_pos) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= m) return;
  const uint32_t k = mover_slots[t];
  const uint32_t i = __ldg(&perm[k]);
  const uint32_t j = (uint32_t)wprefix[i >> 5] + (uint32_t)__popc(mask[i >> 5] & ((1u << (i & 31)) - 1u));
  slot_by_rank[j] = k;
  mover_pos[j] = pos[k];
}

// movers in (new cell, original index) order: old slot and original index
__global__ void __launch_bounds__(256) k_mover_index(const uint32_t* __restrict__ perm_m, int64_t m,
                                                      const uint32_t* __restrict__ slot_by_rank, const uint32_t* __restrict__ perm,
                                                      uint32_t* __restrict__ slot_sorted, uint32_t* __restrict__ idx_sorted) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= m) return;
  const uint32_t k = slot_by_rank[perm_m[r]];
  slot_sorted[r] = k;
  idx_sorted[r] = __ldg(&perm[k]);
}

__device__ __forceinline__ uint32_t lower_bound_u32(const uint32_t* __restrict__ a, uint32_t lo, uint32_t hi, uint32_t x) {
  while (lo < hi) {
    const uint32_t mid = lo + ((hi - lo) >> 1);
    if (__ldg(&a[mid]) < x) lo = mid + 1; else hi = mid;
  }
  return lo;
}

// stayers: to their new slot (relative order kept); the cell id is recomputed from the position
__global__ void __launch_bounds__(256) k_merge_stayers(
    const float4* __restrict__ pos, const float4* __restrict__ vel, const uint32_t* __restrict__ perm,
    const uint32_t* __restrict__ flag_words, const uint32_t* __restrict__ word_prefix, int64_t n, Geometry g,
    const uint32_t* __restrict__ m_start, const uint32_t* __restrict__ m_idx, float4* __restrict__ pos_out,
    float4* __restrict__ vel_out, uint32_t* __restrict__ perm_out) {
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
    const uint32_t fw = __ldg(&flag_words[k >> 5]);
    if ((fw >> (k & 31)) & 1u) continue;                       // a mover: placed by k_merge_movers
    const uint32_t f0 = __ldg(&word_prefix[k >> 5]) + (uint32_t)__popc(fw & ((1u << (k & 31)) - 1u));
    const float4 x = pos[k];
    const uint32_t c = cell_key(x, g), i = __ldg(&perm[k]);
    const uint32_t lo = __ldg(&m_start[c]), hi = __ldg(&m_start[c + 1]);
    const uint32_t at = lo == hi ? lo : lower_bound_u32(m_idx, lo, hi, i);
    const size_t dst = (size_t)k - f0 + at;
    pos_out[dst] = x;
    vel_out[dst] = vel[k];
    perm_out[dst] = i;
  }
}

// movers, in (new cell, original index) order
__global__ void __launch_bounds__(256) k_merge_movers(
    const float4* __restrict__ pos, const float4* __restrict__ vel, const uint32_t* __restrict__ perm,
    const uint32_t* __restrict__ flag_words, const uint32_t* __restrict__ word_prefix, int64_t n,
    const uint32_t* __restrict__ cell_start, int64_t m, const uint32_t* __restrict__ m_key,
    const uint32_t* __restrict__ m_idx, const uint32_t* __restrict__ m_slot, const float4* __restrict__ m_pos_sorted,
    float4* __restrict__ pos_out,
    float4* __restrict__ vel_out, uint32_t* __restrict__ perm_out) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= m) return;
  const uint32_t c = m_key[r], i = m_idx[r], src = m_slot[r];
  const uint32_t p = lower_bound_u32(perm, __ldg(&cell_start[c]), __ldg(&cell_start[c + 1]), i);
  const size_t dst = (size_t)p - movers_before(flag_words, word_prefix, p, (uint32_t)n, (uint32_t)m) + (size_t)r;
  pos_out[dst] = m_pos_sorted[r];          // the movers' sort already carried the positions: no gather through the old slot
  vel_out[dst] = vel[src];
  perm_out[dst] = i;
}

__global__ void __launch_bounds__(256) k_new_cell_start(uint32_t* __restrict__ cell_start, int32_t ncells,
                                                         const uint32_t* __restrict__ flag_words,
                                                         const uint32_t* __restrict__ word_prefix, uint32_t n, uint32_t m,
                                                         const uint32_t* __restrict__ m_start) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c > ncells) return;
  const uint32_t cs = cell_start[c];
  cell_start[c] = cs - movers_before(flag_words, word_prefix, cs, n, m) + __ldg(&m_start[c]);
}

}  // namespace srpp

using namespace srpp;

static inline int ew_grid(const srpp_ctx* c, int64_t n) { return (int)std::min<int64_t>((n + 255) / 256, (int64_t)c->num_sms * 16); }

// scatter the sorted state back to the caller's order
static cudaError_t unsort_state(srpp_ctx* c, int cur, float4* pos_mass, float4* vel, int64_t n) {
  if (n == 0) return cudaSuccess;
  if (n >= kUnsortMinN) {
    // large n: the destinations have no locality; partition by destination instead of scattering (srpp_force.cu A6).
    // Only xyz travel: the caller's arrays still hold the masses / the velocities' .w lanes, which no step changes.
    cudaError_t e = launch_unsort_xyz(c, c->sorted_buf[cur], pos_mass);
    if (e == cudaSuccess) e = launch_unsort_xyz(c, c->vel_s[cur], vel);
    return e;
  }
  k_scatter2_f4<<<ew_grid(c, n), 256, 0, c->stream>>>(c->sorted_buf[cur], c->vel_s[cur], c->perm, n, pos_mass, vel);
  c->launches += 1;
  return cudaGetLastError();
}

extern "C" int32_t srpp_subcycle(srpp_ctx* c, float* pos_mass_f, float* vel_f, float* acc_f, float dt, float kdt, int32_t nsub,
                                 int64_t n) {
  if (!c || n < 0 || n >= ((int64_t)1 << 31) || nsub < 0 || !isfinite(dt) || !isfinite(kdt) ||
      (n > 0 && (!pos_mass_f || !vel_f || !acc_f)) || ((uintptr_t)pos_mass_f & 15u) || ((uintptr_t)vel_f & 15u) ||
      ((uintptr_t)acc_f & 15u))
    return SRPP_ERR_INVALID_ARG;
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return SRPP_ERR_CUDA;
  if (dev != c->device) return SRPP_ERR_STATE;
  float4* pos_mass = (float4*)pos_mass_f;
  float4* vel = (float4*)vel_f;
  float4* acc = (float4*)acc_f;
  cudaStream_t st = c->stream;
  const float half = 0.5f * dt;            // exact in fp32
  auto cuda_fail = [&](cudaError_t e) {
    snprintf(c->cuda_err, sizeof(c->cuda_err), "%s: %s", cudaGetErrorName(e), cudaGetErrorString(e));
    return (int32_t)SRPP_ERR_CUDA;
  };
  int32_t rc;
  cudaError_t e;
  c->rebin_ms_sum = c->subkick_ms_sum = 0.f;
  c->rebin_count = 0;
  if (nsub == 0 || n == 0) return srpp_build_mesh(c, pos_mass_f, n);

  // ---- into sorted space: first half stream in the caller's order, full build, velocities gathered once
  if ((rc = srpp_stream(c, pos_mass_f, vel_f, half, n)) != SRPP_OK) return rc;
  if ((rc = srpp_build_mesh(c, pos_mass_f, n)) != SRPP_OK) return rc;
  int cur = 0;                              // sorted_buf[cur], vel_s[cur], keys_buf[cur] hold the current state
  k_gather_f4<<<ew_grid(c, n), 256, 0, st>>>(vel, c->perm, n, c->vel_s[cur]);
  c->launches += 1;
  const bool incremental_ok = n < ((int64_t)1 << 29);       // the bit-mask scan handles < 2^24 words
  const int ntile = (int)((n + kSubTile - 1) / kSubTile);
  const int64_t nwords = n / 32 + 1;
  SubCounters* ctr = (SubCounters*)((char*)c->m_flags + 128);      // tail of the movers' flag block
  if (c->timing && !c->ev_sub[0]) { cudaEventCreate(&c->ev_sub[0]); cudaEventCreate(&c->ev_sub[1]); }

  for (int32_t s = 0; s < nsub; ++s) {
    const bool last = s == nsub - 1;
    if ((e = launch_accel_sorted(c)) != cudaSuccess) return cuda_fail(e);
    if (last && (e = launch_write_back(c, acc)) != cudaSuccess) return cuda_fail(e);     // caller's order, this mesh's perm
    // ---- kick + stream(s) + new cells + mover detection, one coalesced pass
    if ((e = cudaMemsetAsync(c->mover_mask, 0, 4 * (size_t)nwords, st)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaMemsetAsync(ctr, 0, sizeof(SubCounters), st)) != cudaSuccess) return cuda_fail(e);
    if (c->timing) cudaEventRecord(c->ev_sub[0], st);
    k_kick_stream<<<ntile, kSubThreads, 0, st>>>(c->sorted_buf[cur], c->vel_s[cur], c->acc64, c->perm, n, c->geo,
                                                 c->uniform_mass ? c->mass0 : 1.0f, kdt, half, last ? 0 : 1, c->flag_words,
                                                 c->mover_mask, c->mover_slots, c->m_cap, c->tile_movers, ctr);
    if (c->timing) cudaEventRecord(c->ev_sub[1], st);
    c->launches += 1;
    unsigned long long m_host = 0;
    if ((e = cudaMemcpyAsync(&m_host, &ctr->movers, 8, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e);
    if (c->timing) { float ms = 0.f; cudaEventElapsedTime(&ms, c->ev_sub[0], c->ev_sub[1]); c->subkick_ms_sum += ms; }
    const int64_t m = (int64_t)m_host;
    c->last_movers = (uint64_t)m;
    if (m == 0) continue;                                       // nobody changed cell: the mesh is still right

    if (!incremental_ok || m > c->m_cap) {
      // ---- fall back: back to the caller's order, full build, velocities gathered again
      if ((e = unsort_state(c, cur, pos_mass, vel, n)) != cudaSuccess) return cuda_fail(e);
      if ((rc = srpp_build_mesh(c, pos_mass_f, n)) != SRPP_OK) return rc;
      cur = 0;
      k_gather_f4<<<ew_grid(c, n), 256, 0, st>>>(vel, c->perm, n, c->vel_s[cur]);
      c->launches += 1;
      c->rebin_full += 1;
      continue;
    }

    // ---- incremental re-bin
    if (c->timing) cudaEventRecord(c->ev_sub[0], st);
    // movers ranked by original index -> gathered -> sorted by new cell (stable): (new cell, original index) order
    k_popc_words<<<(int)((nwords + 255) / 256), 256, 0, st>>>(c->mover_mask, nwords, c->mover_wprefix);
    if ((e = launch_scan_u64(st, c->mover_wprefix, (int)nwords, c->sub_scan_tmp, &ctr->pad[0], &ctr->pad[1])) != cudaSuccess) return cuda_fail(e);
    k_mover_place<<<(int)((m + 255) / 256), 256, 0, st>>>(c->mover_slots, m, c->perm, c->mover_mask, c->mover_wprefix,
                                                         c->sorted_buf[cur], c->mover_slot_by_rank, c->mover_pos);
    SortBufs sb;
    sb.flags = c->m_flags; sb.ctl = c->m_ctl; sb.status = c->m_status; sb.status_n = &c->status_n_movers;
    sb.out_sorted = c->m_sorted; sb.tmp_pos = c->m_tmp; sb.vals[0] = c->m_vals[0]; sb.vals[1] = c->m_vals[1];
    sb.keys_out = c->m_keys; sb.cell_start = c->m_cell_start; sb.perm = nullptr;
    // (sort_by_cell clears only the DevFlags part of its flag block: the counters live in the tail)
    if ((e = sort_by_cell(c, sb, c->mover_pos, m)) != cudaSuccess) return cuda_fail(e);
    k_mover_index<<<(int)((m + 255) / 256), 256, 0, st>>>(sb.perm, m, c->mover_slot_by_rank, c->perm, c->mover_slot_sorted,
                                                         c->mover_idx_sorted);
    // F = exclusive prefix of the mover flags over the old slots, kept per 32-slot flag word
    if ((e = launch_scan_u64(st, c->tile_movers, ntile, c->sub_scan_tmp, &ctr->pad[0], &ctr->pad[1])) != cudaSuccess) return cuda_fail(e);
    const int64_t nfw = (n + 31) / 32;
    k_word_prefix<<<(ntile + 7) / 8, 256, 0, st>>>(c->flag_words, nfw, c->tile_movers, c->prefix_f);
    // merge into the other buffer set
    uint32_t* perm_new = c->perm != c->vals_alt ? c->vals_alt : c->vals[0];
    k_merge_stayers<<<ew_grid(c, n), 256, 0, st>>>(c->sorted_buf[cur], c->vel_s[cur], c->perm, c->flag_words, c->prefix_f, n, c->geo,
                                                  c->m_cell_start, c->mover_idx_sorted, c->sorted_buf[cur ^ 1], c->vel_s[cur ^ 1],
                                                  perm_new);
    k_merge_movers<<<(int)((m + 255) / 256), 256, 0, st>>>(c->sorted_buf[cur], c->vel_s[cur], c->perm, c->flag_words, c->prefix_f, n,
                                                          c->cell_start, m, c->m_keys, c->mover_idx_sorted, c->mover_slot_sorted, c->m_sorted,
                                                          c->sorted_buf[cur ^ 1], c->vel_s[cur ^ 1], perm_new);
    k_new_cell_start<<<(c->geo.ncells + 1 + 255) / 256, 256, 0, st>>>(c->cell_start, c->geo.ncells, c->flag_words, c->prefix_f,
                                                                     (uint32_t)n, (uint32_t)m, c->m_cell_start);
    c->launches += 13;
    cur ^= 1;
    c->sorted = c->sorted_buf[cur];
    c->sorted_keys = nullptr;           // the sorted cell ids are not maintained by the merge (nothing reads them)
    c->perm = perm_new;
    c->rebin_incremental += 1;
    if (c->timing) {
      cudaEventRecord(c->ev_sub[1], st);
      if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e);
      float ms = 0.f;
      cudaEventElapsedTime(&ms, c->ev_sub[0], c->ev_sub[1]);
      c->rebin_ms_sum += ms;
      c->rebin_count += 1;
    }
  }
  // ---- back to the caller's order; the context's mesh is the mesh of the returned positions
  if ((e = unsort_state(c, cur, pos_mass, vel, n)) != cudaSuccess) return cuda_fail(e);
  if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e);
  return SRPP_OK;
}
