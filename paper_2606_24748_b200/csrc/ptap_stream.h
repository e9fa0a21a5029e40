// ptap_stream.h -- device-side view of a StreamPlan (internal.h) and the launcher of the staged product kernels.
#pragma once
#include "internal.h"

namespace bsramg {

constexpr int STREAM_THREADS_DIRECT = 256;           // stage 1: 8 warps per brick, two bricks per SM
constexpr int STREAM_MINB1 = 2;
constexpr int STREAM_THREADS_PERSIST = 128;          // stage 2: 4 warps per coarse row (36 accumulators per lane)
constexpr int64_t STREAM_SMEM_BUDGET = 112 * 1024;   // dynamic shared memory a brick may use (2 x (112+1) KB <= 228 KB)
constexpr int64_t STREAM_SMEM_BUDGET_PERSIST = 75000;  // stage 2: three coarse rows per SM (register-limited)

struct StreamArgs {  // all device pointers
  const StreamBrickHdr* bricks;
  const StreamChunkHdr* chunks;
  const StreamRun *xruns, *yruns;
  const StreamEntry* entries;
  const StreamPass* passes;
  const StreamMeta* meta;
  const double *xvals, *yvals;
  double* cvals;
};

// device copy of a StreamPlan
struct StreamDev {
  bool ok = false, persist = false;
  int64_t nbricks = 0, smem = 0, bytes = 0;
  StreamArgs args{};
  std::vector<void*> owned;
};

int stream_upload(const StreamShape& sh, const StreamPlan& sp, StreamDev& sd, cudaStream_t st);
void stream_release(StreamDev& sd);
// prepare = true: cold call that sets the kernel's dynamic shared memory attribute on the current device
int stream_launch(int M, int K, int N, const StreamArgs& a, bool persist, int64_t nbricks, int64_t smem, cudaStream_t st,
                  bool prepare = false);

}  // namespace bsramg
