// srpp_internal.cuh -- context, workspace layout and launch declarations shared by the CUDA
// translation units of libsrpp (product path only; the CPU oracle shares nothing with this).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#include "srpp.h"

namespace srpp {

// ---- tunables ------------------------------------------------------------------------------
// binning: LSD counting sort of the cell id in digits of <= 8 bits, payload carried (srpp_mesh.cu)
constexpr int kSortThreads = 512;             // 16 warps
constexpr int kSortWarps = kSortThreads / 32;
constexpr int kSortItems = 8;                 // a warp handles 8 steps of 32 consecutive elements
constexpr int kSortTile = kSortThreads * kSortItems;  // 4096 elements per tile
#ifndef SRPP_PASS_TILE
#define SRPP_PASS_TILE 4096
#endif
constexpr int kPassTile = SRPP_PASS_TILE;     // elements per tile of a digit pass (k_sort_pass)
constexpr int kSortMinDigitBits = 5;          // >= 32 bins (one warp-row of the column scan)
constexpr int kSortMaxDigitBits = 8;          // <= 256 bins: >= 16 elements per bin and tile, so the per-digit runs cover whole 32-byte sectors
constexpr int kSortMaxBins = 1 << kSortMaxDigitBits;
constexpr int kSortMaxPasses = 3;             // 3 x 8 bits cover the 2^24-cell limit
// sort control block: 64 words of tile tickets (one per pass) + the global digit histograms [passes][kSortMaxBins]
constexpr size_t sort_ctl_bytes() { return sizeof(uint32_t) * (64 + (size_t)kSortMaxPasses * kSortMaxBins); }

#ifndef SRPP_FORCE_THREADS
#define SRPP_FORCE_THREADS 256
#endif
constexpr int kForceThreads = SRPP_FORCE_THREADS;   // 8 autonomous warps per CTA
constexpr int kForceWarps = kForceThreads / 32;
#ifndef SRPP_SRC_TILE
#define SRPP_SRC_TILE 128
#endif
#ifndef SRPP_SRC_CHUNK
#define SRPP_SRC_CHUNK 1024
#endif
constexpr int kSrcTile = SRPP_SRC_TILE;       // sources staged per warp-private smem tile (float4 each)
constexpr int kSrcChunk = SRPP_SRC_CHUNK;     // sources per work item (fp32 partial-sum length)
constexpr int kMaxSeg = 18;                   // 9 (dy,dz) rows x up to 2 x-segments (periodic wrap)
constexpr int64_t kUnsortMinN = (int64_t)1 << 22;   // write-back: below this acc and vel sit in L2 and the direct scatter wins
// run cursors of the bucketed write-back: one per bucket of every level (at most 256 + 65536 + n/4096 + 3)
constexpr size_t unsort_cursor_bytes(int64_t n) { return sizeof(uint32_t) * ((size_t)(n > 0 ? n : 1) / 4096 + 65536 + 256 + 8); }

// timing events: mesh begin/end, accel begin, force-kernel begin/end, accel end
enum { kEvMesh0 = 0, kEvMesh1, kEvAccel0, kEvForce0, kEvForce1, kEvAccel1, kNumEvents };

// ---- device-side flag / counter block (first 256 bytes of the workspace) -------------------
struct DevFlags {
  uint32_t domain_error;     // A1 found a position outside [0,L) or non-finite (R13)
  uint32_t mass_nonuniform;  // some particle's mass differs from particle 0's
  uint32_t max_cell_count;
  uint32_t pad0;
  unsigned long long item_counter;    // dynamic work queue head of the force kernel
  unsigned long long total_items;
  unsigned long long candidate_pairs; // W
  unsigned long long pair_slots;
  unsigned long long big_pairs;       // part of W that sits in cells of more than 64 particles (picks the force kernel build)
};

struct Geometry {
  float box[3];
  float inv_cell[3];     // (float)ncell / box, one IEEE fp32 division (R10)
  float cell_w[3];       // box / ncell (fp32), only used to pick integer reference points
  int32_t ncell[3];
  int32_t ncells;
  int32_t periodic[3];   // 1: periodic axis (stencil wraps, image shift); 0: open axis (stencil stops at the faces)
  int32_t act_lo[3];     // cells [act_lo, act_hi) per axis hold the ACTIVE targets; the other cells are passive
  int32_t act_hi[3];     //   (sources only) -- the overloaded node volume of PAPER.md:65/73
};

struct ForceConst {
  float eps2;            // eps^2 rounded to fp32: seeds the s-FMA chain, u = s + eps2
  float rc2e;            // rc^2 + eps2: cutoff test on u
  float nq[6];           // -Q(u) coefficients, Q(u) = P(u - eps2), expanded in fp64
  float pad;             // coordinate of padded (empty) target / source slots: beyond rc of every real one at any scale
  int32_t fine_items;    // tiny problem: 16-target items so that every resident warp gets work
};

#ifdef __CUDACC__
// A1 (R10, R11): one IEEE multiply per axis (never contracted: there is nothing to fuse with), floor, clamp.
__device__ __forceinline__ uint32_t cell_key(const float4& p, const Geometry& g) {
  int cx = (int)floorf(__fmul_rn(p.x, g.inv_cell[0]));
  int cy = (int)floorf(__fmul_rn(p.y, g.inv_cell[1]));
  int cz = (int)floorf(__fmul_rn(p.z, g.inv_cell[2]));
  cx = max(min(cx, g.ncell[0] - 1), 0);       // the lower clamp only matters for inputs that already raised DOMAIN
  cy = max(min(cy, g.ncell[1] - 1), 0);
  cz = max(min(cz, g.ncell[2] - 1), 0);
  return (uint32_t)cx + (uint32_t)g.ncell[0] * ((uint32_t)cy + (uint32_t)g.ncell[1] * (uint32_t)cz);
}

__device__ __forceinline__ bool in_domain(const float4& p, const Geometry& g) {
  return (p.x >= 0.f) && (p.x < g.box[0]) && (p.y >= 0.f) && (p.y < g.box[1]) && (p.z >= 0.f) && (p.z < g.box[2]);
}

// stream wrap (R13, R17): one box length at most; a value that rounds to L becomes 0
__device__ __forceinline__ float wrap_coord(float y, float L) {
  if (y >= L) y -= L;
  else if (y < 0.f) y += L;
  if (!(y < L)) y = 0.f;
  return y;
}

#endif

}  // namespace srpp

struct srpp_ctx {
  srpp_params params;
  srpp::Geometry geo;
  srpp::ForceConst fc;
  cudaStream_t stream;
  int device;
  int num_sms;
  int force_blocks_per_sm[2];   // resident CTAs per SM of the two builds of the force kernel
  int64_t n_capacity;        // particles the workspace was sized for (== n of build_mesh)
  int64_t n;                 // particles of the last successful build_mesh, -1 before
  int sort_passes;           // digits of the cell id (LSD passes)
  int sort_digit_bits;       // bits per digit
  int sort_blocks;
  int sort_blocks_per_sm;
  bool sort_attr_set;
  bool unsort_attr_set;
  uint32_t* unsort_cursor;   // run cursors of the bucketed write-back (srpp_force.cu), unsort_cursor_bytes(n)
  bool uniform_mass;
  float mass0;
  // workspace carve-up (device pointers)
  char* ws;
  size_t ws_bytes;
  srpp::DevFlags* flags;
  uint32_t* vals[2];         // original indices, ping-pong (unequal masses) / perm of the last pass
  uint32_t* vals_alt;        // third index buffer: the incremental re-bin writes the new perm beside the current one
  uint32_t* keys_buf[2];     // cell ids in sorted order: [0] written by a full build, [1] its ping-pong partner
  float4* sorted_buf[2];     // sorted positions: [0] written by a full build, [1] ping-pong partner of the re-bin
  float4* vel_s[2];          // velocities in sorted order (srpp_subcycle), ping-pong
  uint32_t* prefix_f;        // [n/32+2] movers in the slots before each 32-slot flag word
  uint32_t* flag_words;      // [n/32+2] bit k&31 of word k>>5: the particle in sorted slot k changed cell
  uint32_t* mover_mask;      // [n/32+1] bit i set: particle with original index i changed cell
  unsigned long long* mover_wprefix;  // [n/32+2] exclusive prefix of popc(mover_mask)
  unsigned long long* tile_movers;    // [n/1024+2] movers per 1024 sorted slots, scanned in place
  unsigned long long* sub_scan_tmp;   // scan scratch
  uint32_t* mover_slots;     // [m_cap] unordered list of the sorted slots that hold movers
  uint32_t* mover_slot_by_rank;  // [m_cap] slot of the j-th mover in ascending original index
  float4* mover_pos;         // [m_cap] their new positions (input of the movers' sort)
  uint32_t* mover_idx_sorted;    // [m_cap] original index, in (new cell, index) order
  uint32_t* mover_slot_sorted;   // [m_cap] old slot, same order
  // second sort buffer set (the movers)
  srpp::DevFlags* m_flags; uint32_t* m_ctl; unsigned long long* m_status; float4* m_sorted; float4* m_tmp;
  uint32_t* m_vals[2]; uint32_t* m_keys; uint32_t* m_cell_start;
  int64_t status_n_movers;
  int64_t m_cap;             // movers the second set is sized for (n/4): beyond it the re-bin falls back to a full build
  uint64_t rebin_incremental, rebin_full, last_movers;   // counters (srpp_get_stats)
  cudaStream_t copy_stream;  // srpp_step_host: second stream for the copies that overlap the kernels
  cudaEvent_t ev_copy[3];
  cudaEvent_t ev_sub[2];     // timing of the re-bins inside srpp_subcycle
  float rebin_ms_sum, subkick_ms_sum; int rebin_count;
  uint32_t* sort_ctl;        // tile tickets + global digit histograms (cleared by every build)
  unsigned long long* sort_status;  // [tiles][kSortMaxBins] look-back status words, epoch-tagged
  int64_t status_n;          // n the status array was last cleared for (0 = never)
  uint32_t sort_epoch;       // tag of the last pass launched
  float4* pos_tmp;           // payload ping-pong buffer (aliases acc64: mesh build and accel never overlap)
  uint32_t* cell_start;      // [ncells+1]
  float4* sorted;            // [n] current sorted positions (== sorted_buf[0] after a full build)
  unsigned long long* item_prefix;  // [ncells+1] exclusive prefix of per-cell work items
  unsigned long long* scan_tmp;     // block sums for the 64-bit scan
  double* acc64;             // [3n] fp64 accumulators, sorted order
  const uint32_t* perm;      // == vals[(sort_passes - 1) & 1]
  const uint32_t* sorted_keys;
  srpp::DevFlags flags_host; // last read-back
  char cuda_err[256];
  // optional per-phase device timing (srpp_set_timing): events recorded on `stream` around the phases
  bool timing;
  cudaEvent_t ev[srpp::kNumEvents];
  bool ev_mesh_valid, ev_accel_valid;
  uint64_t launches;         // kernels launched by this context so far (harness evidence)
  int mbp_occ;               // resident CTAs per SM of k_mbp_phi (queried once)
  void* block_plan;          // srpp_blocks.cu: x-partition + last timings (host), nullptr until srpp_blocks_init
};

namespace srpp {

// buffer set of one sort_by_cell call
struct SortBufs {
  DevFlags* flags; uint32_t* ctl; unsigned long long* status; int64_t* status_n;
  float4* out_sorted; float4* tmp_pos; uint32_t* vals[2]; uint32_t* keys_out; uint32_t* cell_start;
  uint32_t* perm;            // result: == vals[(passes - 1) & 1]
};

size_t workspace_layout(const srpp_params& p, int64_t n, srpp_ctx* ctx /*nullable: fill pointers*/);

// srpp_mesh.cu
cudaError_t launch_build_mesh(srpp_ctx* c, const float4* pos_mass, int64_t n);
cudaError_t sort_by_cell(srpp_ctx* c, SortBufs& sb, const float4* pos_mass, int64_t n);
void plan_sort(int32_t ncells, int* passes, int* digit_bits);
// srpp_force.cu
// force + write-back (+ the kick of A7 fused into the write-back when vel != nullptr)
cudaError_t launch_accel(srpp_ctx* c, float4* acc, float4* vel = nullptr, float kdt = 0.f);
cudaError_t launch_accel_sorted(srpp_ctx* c);                  // force only: fp64 accumulators in sorted order
cudaError_t launch_write_back(srpp_ctx* c, float4* acc, float4* vel = nullptr, float kdt = 0.f);   // A6 (+ A7)
cudaError_t launch_unsort_xyz(srpp_ctx* c, const float4* sorted_src, float4* dst);   // bucketed scatter of xyz through perm
// srpp_subcycle.cu
cudaError_t launch_subcycle(srpp_ctx* c, float4* pos_mass, float4* vel, float4* acc, float dt, float kdt, int nsub,
                            int64_t n, int32_t* status_out);
cudaError_t launch_kick(srpp_ctx* c, float4* vel, const float4* acc, float kdt, int64_t n);
cudaError_t launch_stream(srpp_ctx* c, float4* pos_mass, const float4* vel, float dt, int64_t n);
void query_force_occupancy(int* blocks_per_sm /*[2]*/);
// in-place exclusive scan of data[0..n) (n <= 2^24); the total goes to *total_out and *total_out2 (device pointers)
cudaError_t launch_scan_u64(cudaStream_t st, unsigned long long* data, int n, unsigned long long* tmp,
                            unsigned long long* total_out, unsigned long long* total_out2);
// srpp_mbp.cu
size_t mbp_workspace_layout(int64_t n, int64_t nhalo, size_t* o_phi, size_t* o_prefix, size_t* o_start, size_t* o_tmp);
cudaError_t launch_mbp(srpp_ctx* c, const float4* pos_mass, int64_t n, const int64_t* halo_start_host, int64_t nhalo,
                       float* phi_out, long long* mbp_index, float* mbp_phi, char* ws);
// srpp_blocks.cu
void free_block_plan(srpp_ctx* c);
// srpp_probe.cu
cudaError_t run_fp32_probe(cudaStream_t st, int variant, int iters, double* flops_per_s, float* checksum);

}  // namespace srpp
