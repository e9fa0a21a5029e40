// ptap_stream.h -- device-side view of a StreamPlan (internal.h) and the launcher of the stream kernels.
#pragma once
#include "internal.h"

namespace bsramg {

constexpr int STREAM_THREADS = 256;                  // 8 warps per brick; two bricks per SM
constexpr int64_t STREAM_SMEM_BUDGET = 112 * 1024;   // dynamic shared memory a brick may use (2 x (112+1) KB <= 228 KB)

struct StreamArgs {  // all device pointers
  const int32_t *br_chunk_ptr, *br_acc_ptr, *acc_slot;
  const int32_t *ch_xrun_ptr, *ch_yrun_ptr, *ch_item_ptr, *ch_red_ptr, *ch_gptr, *ch_nx, *ch_ny, *ch_nparts;
  const int64_t* ch_code_ptr;
  const StreamRun *xruns, *yruns;
  const StreamItem* items;
  const StreamRed* reds;
  const void* codes;
  const double *xvals, *yvals;
  double* cvals;
};

// device copy of a StreamPlan
struct StreamDev {
  bool ok = false, wide = false;
  int64_t nbricks = 0, smem = 0, bytes = 0;
  StreamArgs args{};
  std::vector<void*> owned;
};

int stream_groups(int N);
int stream_upload(const StreamPlan& sp, StreamDev& sd, cudaStream_t st);
void stream_release(StreamDev& sd);
int stream_launch(int M, int K, int N, const StreamArgs& a, bool wide, int64_t nbricks, int64_t smem, cudaStream_t st);

}  // namespace bsramg
