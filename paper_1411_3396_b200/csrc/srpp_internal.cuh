// srpp_internal.cuh -- context, workspace layout and launch declarations shared by the CUDA
// translation units of libsrpp (product path only; the CPU oracle shares nothing with this).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#include "srpp.h"

namespace srpp {

// ---- tunables ------------------------------------------------------------------------------
constexpr int kRadixBits = 8;                 // LSD radix digit width (A2-A4 as digit-wise counting sort)
constexpr int kRadix = 1 << kRadixBits;
constexpr int kSortThreads = 256;             // 8 warps
constexpr int kSortKeysPerThread = 8;         // warp handles 8 steps of 32 consecutive keys
constexpr int kSortTile = kSortThreads * kSortKeysPerThread;  // 2048 keys per tile
constexpr int kSortBlocksPerSM = 4;

constexpr int kForceThreads = 256;            // 8 autonomous warps per CTA
constexpr int kForceWarps = kForceThreads / 32;
constexpr int kSrcTile = 128;                 // sources staged per warp-private smem tile (64 pairs)
constexpr int kSrcChunk = 1024;               // sources per work item (fp32 partial-sum length)
constexpr int kMaxSeg = 18;                   // 9 (dy,dz) rows x up to 2 x-segments (periodic wrap)

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
};

struct Geometry {
  float box[3];
  float inv_cell[3];     // (float)ncell / box, one IEEE fp32 division (R10)
  float cell_w[3];       // box / ncell (fp32), only used to pick integer reference points
  int32_t ncell[3];
  int32_t ncells;
};

struct ForceConst {
  float eps2;            // eps^2 rounded to fp32: seeds the s-FMA chain, u = s + eps2
  float rc2e;            // rc^2 + eps2: cutoff test on u
  float nq[6];           // -Q(u) coefficients, Q(u) = P(u - eps2), expanded in fp64
};

}  // namespace srpp

struct srpp_ctx {
  srpp_params params;
  srpp::Geometry geo;
  srpp::ForceConst fc;
  cudaStream_t stream;
  int device;
  int num_sms;
  int force_blocks_per_sm;
  int64_t n_capacity;        // particles the workspace was sized for (== n of build_mesh)
  int64_t n;                 // particles of the last successful build_mesh, -1 before
  int sort_passes;
  int sort_blocks;
  bool uniform_mass;
  float mass0;
  // workspace carve-up (device pointers)
  char* ws;
  size_t ws_bytes;
  srpp::DevFlags* flags;
  uint32_t* keys[2];
  uint32_t* vals[2];
  uint32_t* hist;            // [kRadix][sort_blocks]
  uint32_t* cell_start;      // [ncells+1]
  float4* sorted;            // [n]
  unsigned long long* item_prefix;  // [ncells+1] exclusive prefix of per-cell work items
  unsigned long long* scan_tmp;     // block sums for the 64-bit scan
  double* acc64;             // [3n] fp64 accumulators, sorted order
  const uint32_t* perm;      // == vals[sort_passes & 1]
  const uint32_t* sorted_keys;
  srpp::DevFlags flags_host; // last read-back
  char cuda_err[256];
  // optional per-phase device timing (srpp_set_timing): events recorded on `stream` around the phases
  bool timing;
  cudaEvent_t ev[srpp::kNumEvents];
  bool ev_mesh_valid, ev_accel_valid;
  uint64_t launches;         // kernels launched by this context so far (harness evidence)
};

namespace srpp {

size_t workspace_layout(const srpp_params& p, int64_t n, srpp_ctx* ctx /*nullable: fill pointers*/);

// srpp_mesh.cu
cudaError_t launch_build_mesh(srpp_ctx* c, const float4* pos_mass, int64_t n);
// srpp_force.cu
cudaError_t launch_accel(srpp_ctx* c, float4* acc);
cudaError_t launch_kick(srpp_ctx* c, float4* vel, const float4* acc, float kdt, int64_t n);
cudaError_t launch_stream(srpp_ctx* c, float4* pos_mass, const float4* vel, float dt, int64_t n);
int query_force_occupancy();
// srpp_probe.cu
cudaError_t run_fp32_probe(cudaStream_t st, int variant, int iters, double* flops_per_s, float* checksum);

}  // namespace srpp
