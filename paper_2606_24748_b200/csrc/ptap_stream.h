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
  // store epilogue of prolongator smoothing (smooth.cu; direct bricks only): C(row,J) = own(row,J) - omega * D_row^-1 * acc
  const double* dinv = nullptr;       // M x M per X row
  const double* own_vals = nullptr;   // blocks of the tentative prolongator
  const int32_t* out_row = nullptr;   // per output slot: its row
  const int32_t* own_slot = nullptr;  // per output slot: the tentative block with the same coordinate, or -1
  double omega = 0.0;
  int32_t brick0 = 0;                 // first brick of this launch (a plan may be launched in several pieces)
};

// device copy of a StreamPlan
struct StreamDev {
  bool ok = false, persist = false;
  int64_t nbricks = 0, smem = 0, bytes = 0;
  StreamArgs args{};
  std::vector<void*> owned;
  // host copies for the chunked host-buffer path: the largest X row every leading run of bricks needs (direct plans)
  // and, for persist plans, the end of every brick's output in C slots
  std::vector<int32_t> brick_maxrow_prefix, brick_out_end;
};

int stream_upload(const StreamShape& sh, const StreamPlan& sp, StreamDev& sd, cudaStream_t st, bool smooth = false);
void stream_release(StreamDev& sd);
// prepare = true: cold call that sets the kernel's dynamic shared memory attribute on the current device
int stream_launch(int M, int K, int N, const StreamArgs& a, bool persist, int64_t nbricks, int64_t smem, cudaStream_t st,
                  bool prepare = false);
// the direct kernel with the smoothing epilogue (shapes <2,2,3>, <3,3,3>, <3,3,6>, <6,6,6>)
int stream_launch_smooth(int M, int N, const StreamArgs& a, int64_t nbricks, int64_t smem, cudaStream_t st,
                         bool prepare = false);

}  // namespace bsramg
