// =============================================================================================
// tpc_prof.cuh -- launch accounting and optional per-kernel CUDA-event timing on the LAUNCHING
// stream (bench.py's `roofline` and `gpu_launches`; include/tpc_b200.h tpc_profile_*).
//
// Every kernel launch of the library goes through TPC_LAUNCH(id, stream, kernel<<<...>>>(...)):
//   - the per-kernel launch counter is always incremented (host side, a few ns);
//   - when profiling is enabled, a cudaEvent pair is recorded around the launch on the same
//     stream; tpc_profile_collect() later synchronises those events and sums the elapsed times
//     per kernel id.  Disabled (the default) it costs nothing on the device.
// Not thread-safe: one host thread drives one GPU ("one CPU core per GPU").
// =============================================================================================
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tpc {

enum KernelId {
  KID_BUCKET_HIST = 0,
  KID_SCAN,
  KID_PART_SCATTER,
  KID_BUCKET_SCATTER,
  KID_BUCKET_SORT,
  KID_NEIGHBOURS,
  KID_CLEAN,
  KID_COMPACT_STARTS,
  KID_FOLLOW,
  KID_SURVIVORS,
  KID_FOLLOW_B,
  KID_PUSH_KEYS,
  KID_COUNT_KEPT,
  KID_WRITE_TRACKS,
  KID_ASSIGN,
  KID_FIT,
  KID_TRACK_TIME,
  KID_COLLISIONS,
  KID_MERGE,
  KID_CLUSTERIZE,
  KID_FIT_PHYSICS,
  KID_EXPORT,
  KID_N
};

void prof_begin(int id, cudaStream_t st);
void prof_end(int id, cudaStream_t st);
// Counts one launch of kernel `id` and nothing else: no event is created or recorded, whatever tpc_profile_enable
// says.  For entry points that promise to allocate nothing (tpc_pair_sides_static).
void prof_count(int id);

struct ProfScope {
  int id;
  cudaStream_t st;
  ProfScope(int i, cudaStream_t s) : id(i), st(s) { prof_begin(id, st); }
  ~ProfScope() { prof_end(id, st); }
};

}  // namespace tpc

#define TPC_LAUNCH(id, st, ...)       \
  do {                                \
    ::tpc::ProfScope _ps((id), (st)); \
    __VA_ARGS__;                      \
  } while (0)
