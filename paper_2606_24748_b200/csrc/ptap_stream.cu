// ptap_stream.cu -- the hot kernels of ptap_numeric: brick-staged, output-stationary, k-synchronous block products.
//
// PAPER.md:219 (the dominant kernel is the numeric A*P with block sizes <3,3,6>), PAPER.md:103 ("local blocked triple
// product"), PAPER.md:97-99, 248-250 (coarse blocks summed through a precomputed block plan, contiguous bs_r*bs_c
// runs).  Schedule format: internal.h / ptap_stream.cpp.
//
// One CTA = one brick.  Per chunk it stages the X blocks (A rows / a piece of an R row), every Y row they reference
// (P rows / AP rows) and the per-block masks in shared memory: runs of 16-byte-multiple blocks by TMA bulk copies
// (cp.async.bulk, bytes counted on an mbarrier), padded 3x3 blocks and the small tables by cp.async.  A lane owns one
// output block (M x N accumulators in registers); its warp walks the X blocks of the row in order.  At step k all
// lanes of a row read X(row,k) -- one shared-memory broadcast -- and the lanes whose bit is set in the block's mask
// read consecutive blocks of Y's row, so every shared-memory access is a broadcast or contiguous (the gathers that
// made the one-thread-per-block version L1-bound, profiles/r1a_first_path.md, are gone) and HBM sees each operand
// once per brick (Y again from L2 for neighbouring bricks).  No atomics: stage 1 writes each AP block once from
// registers; stage 2 adds the warps' partial coarse blocks in warp order through shared memory and writes each A_c
// block once.
#include "internal.h"
#include "ptap_stream.h"

namespace bsramg {

__device__ __forceinline__ int64_t up16d(int64_t b) { return (b + 15) & ~int64_t(15); }

// asynchronous global -> shared copies (LDGSTS): every thread issues all of its copies back to back and the CTA
// waits once, so a chunk pays the memory latency once instead of once per loop trip
template <int BYTES>
__device__ __forceinline__ void cp_async(void* dst_smem, const void* src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(dst_smem);
  if (BYTES == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(src));
  else if (BYTES == 8) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(src));
  else asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(src));
}
__device__ __forceinline__ void cp_async_wait_all() {
  asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
}

// ---- bulk (TMA) copies: one thread moves a whole run of blocks global -> shared; completion is counted in bytes on
// an mbarrier.  Used for every operand whose blocks are a multiple of 16 bytes (everything but 3x3 X blocks, which
// are padded on the way in); the shared-memory side is written in full lines by the copy engine instead of one
// 16-byte LDGSTS wavefront per sector (profiles/r1g_final.md: 11.5 wavefronts per 512-byte LDGSTS.128).
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count));
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("{ .reg .b64 st; mbarrier.arrive.shared::cta.b64 st, [%0]; }" ::"r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned phase) {
  unsigned done;
  do {
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(done) : "r"((unsigned)__cvta_generic_to_shared(bar)), "r"(phase) : "memory");
  } while (!done);
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src, unsigned bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"((unsigned)__cvta_generic_to_shared(dst_smem)), "l"(src), "r"(bytes),
                 "r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

}  // namespace bsramg
namespace bsramg {
// cold: opts `kern` in to the device's largest dynamic shared memory size.  The attribute belongs to the kernel, not
// to a plan: it is always raised to the device limit, so that plans of different sizes (or built on different
// threads) never lower it for one another; what a launch uses is the plan's own size.
template <typename K>
static int optin_shared_memory(K kern, int64_t need) {
  int dev = 0, lim = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  CUDA_TRY(cudaDeviceGetAttribute(&lim, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
  cudaFuncAttributes fa;
  CUDA_TRY(cudaFuncGetAttributes(&fa, kern));
  lim -= (int)fa.sharedSizeBytes;   // the limit covers static + dynamic shared memory
  if (need > lim) return fail(BSR_ERR_LIMIT, "a brick needs %lld bytes of shared memory, the device offers %d", (long long)need, lim);
  CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, lim));
  return BSR_OK;
}

template <int NE>
__device__ __forceinline__ void lds_block(const double* __restrict__ p, double (&v)[NE]) {  // p 16-byte aligned if NE even
  if (NE % 2 == 0) {
#pragma unroll
    for (int e = 0; e < NE / 2; ++e) {
      const double2 t = reinterpret_cast<const double2*>(p)[e];
      v[2 * e] = t.x;
      v[2 * e + 1] = t.y;
    }
  } else {
#pragma unroll
    for (int e = 0; e < NE; ++e) v[e] = p[e];
  }
}

template <int M, int K, int N, int NT, bool PERSIST, int EPI = 0>
__global__ void __launch_bounds__(NT, PERSIST ? 3 : STREAM_MINB1)
stream_product_kernel(const StreamArgs a) {
  static_assert(EPI == 0 || (!PERSIST && M == K), "the smoothing epilogue belongs to the direct A*P~ product");
  constexpr int MK = M * K, KN = K * N, MN = M * N, XS = (MK + 1) & ~1, NW = NT / 32;
  extern __shared__ __align__(16) unsigned char smem[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int b = blockIdx.x + a.brick0;
  // brick and chunk headers: one 16-byte and one 64-byte broadcast load (a direct brick is its own single chunk, so
  // both loads are issued together)
  const int4 bh = __ldg(reinterpret_cast<const int4*>(a.bricks + b));  // chunk0, nchunks, out, nslots
  const int br_nslots = bh.w;
  constexpr bool XBULK = (MK % 2 == 0), YBULK = (KN % 2 == 0);   // runs of whole 16-byte multiples
  __shared__ uint64_t bulk_bar;
  if (XBULK || YBULK) {
    if (tid == 0) mbar_init(&bulk_bar, NT);
    __syncthreads();
  }

  double acc[MN];
#pragma unroll
  for (int e = 0; e < MN; ++e) acc[e] = 0.0;

  for (int ci = 0; ci < (PERSIST ? bh.y : 1); ++ci) {
    const int ch = PERSIST ? bh.x + ci : b;
    const int4* hp = reinterpret_cast<const int4*>(a.chunks + ch);
    const int4 h0 = __ldg(hp), h1 = __ldg(hp + 1), h2 = __ldg(hp + 2);
    const int64_t meta0 = ((int64_t)(uint32_t)h0.x) | ((int64_t)h0.y << 32);
    const int nx = h0.z, ny = h0.w;
    const int ent0 = h1.x, nent = h1.y, pass0 = h1.z, npass = h1.w;
    const int xr0 = h2.x, nxr = h2.y, yr0 = h2.z, nyr = h2.w;
    const int nmeta = __ldg(reinterpret_cast<const int*>(hp + 3));   // even (padded by the plan)
    double* Xs = reinterpret_cast<double*>(smem);
    StreamMeta* metas = reinterpret_cast<StreamMeta*>(smem + up16d((int64_t)nx * XS * 8));
    double* Ys = reinterpret_cast<double*>(reinterpret_cast<unsigned char*>(metas) + up16d((int64_t)nmeta * 8));
    StreamEntry* entries = reinterpret_cast<StreamEntry*>(reinterpret_cast<unsigned char*>(Ys) + up16d((int64_t)ny * KN * 8));
    StreamPass* passes = reinterpret_cast<StreamPass*>(entries + nent);
    // ---- stage X (padded to XS doubles per block), masks, Y, entries, passes.  Runs are dealt to the warps; a warp
    // fetches the descriptors of up to 32 of its runs with one load per lane (one memory latency for all of them)
    {
      const int nruns = nxr + nyr;  // X runs first
      for (int base = warp; base < nruns; base += NW * 32) {
        const int mine = base + lane * NW;
        StreamRun run = {0, 0, 0};
        const bool have = mine < nruns, isx = mine < nxr;
        if (have) run = isx ? a.xruns[xr0 + mine] : a.yruns[yr0 + (mine - nxr)];
        // runs of 16-byte-multiple blocks: this lane hands its run to the copy engine
        if (have && isx && XBULK && run.n > 0) {
          mbar_expect_tx(&bulk_bar, (unsigned)run.n * MK * 8);
          bulk_g2s(Xs + (int64_t)run.dst * XS, a.xvals + (int64_t)run.src * MK, (unsigned)run.n * MK * 8, &bulk_bar);
        }
        if (have && !isx && YBULK && run.n > 0) {
          mbar_expect_tx(&bulk_bar, (unsigned)run.n * KN * 8);
          bulk_g2s(Ys + (int64_t)run.dst * KN, a.yvals + (int64_t)run.src * KN, (unsigned)run.n * KN * 8, &bulk_bar);
        }
        if ((XBULK || nxr == 0) && YBULK) continue;   // nothing left for the LDGSTS path
        const int cnt = min(32, (nruns - base + NW - 1) / NW);
        for (int t = 0; t < cnt; ++t) {
          const int src = __shfl_sync(0xffffffffu, run.src, t), n = __shfl_sync(0xffffffffu, run.n, t);
          const int dst = __shfl_sync(0xffffffffu, run.dst, t);
          if (base + t * NW < nxr) {
            if (!XBULK) {   // padded blocks: element by element
              const double* gs = a.xvals + (int64_t)src * MK;
              double* sd = Xs + (int64_t)dst * XS;
              for (int e = lane; e < n * MK; e += 32) {
                const int blk = e / MK;
                cp_async<8>(sd + blk * XS + (e - blk * MK), gs + e);
              }
            }
          } else if (!YBULK) {
            const double* gs = a.yvals + (int64_t)src * KN;
            double* sd = Ys + (int64_t)dst * KN;
            for (int e = lane; e < n * KN; e += 32) cp_async<8>(sd + e, gs + e);
          }
        }
      }
    }
    {
      const uint4* msrc = reinterpret_cast<const uint4*>(a.meta + meta0);
      for (int e = tid; e < nmeta / 2; e += NT) cp_async<16>(reinterpret_cast<uint4*>(metas) + e, msrc + e);
      const uint4* esrc = reinterpret_cast<const uint4*>(a.entries + ent0);
      for (int e = tid; e < nent; e += NT) cp_async<16>(reinterpret_cast<uint4*>(entries) + e, esrc + e);
      const uint4* psrc = reinterpret_cast<const uint4*>(a.passes + pass0);
      for (int e = tid; e < npass; e += NT) cp_async<16>(reinterpret_cast<uint4*>(passes) + e, psrc + e);
    }
    cp_async_wait_all();
    if (XBULK || YBULK) {
      mbar_arrive(&bulk_bar);              // every thread has posted the bytes of its runs
      mbar_wait(&bulk_bar, (unsigned)(ci & 1));
    }
    __syncthreads();
    // ---- the passes of this warp
    for (int p = warp; p < npass; p += NW) {
      const StreamPass ps = passes[p];
      int xbase = 0, mbase = 0, len = 0, out = 0, slot = -1;   // slot: inside the entry's window of the row's slots
      for (int e = ps.e0; e < ps.e1; ++e) {
        const StreamEntry en = entries[e];
        const int l0 = en.lane0();
        if (lane >= l0 && lane < l0 + en.nslots()) {
          xbase = en.xbase; mbase = en.mbase; len = en.len(); out = en.out; slot = en.slot0() + lane - l0;
        }
      }
      if (!PERSIST) {
#pragma unroll
        for (int e = 0; e < MN; ++e) acc[e] = 0.0;
      }
      const uint32_t below = slot >= 0 ? ((1u << slot) - 1u) : 0u;
      // the mask of step k+1 is fetched while step k computes (one shared-memory latency off the critical path)
      StreamMeta nxt = metas[mbase];
      for (int k = 0; k < ps.steps; ++k) {
        const StreamMeta mt = nxt;
        nxt = metas[mbase + min(k + 1, max(len - 1, 0))];
        if (slot >= 0 && k < len) {
          if ((mt.mask >> slot) & 1u) {
            const double* xp = Xs + (int64_t)(xbase + k) * XS;
            const double* yp = Ys + (int64_t)(mt.ybase + __popc(mt.mask & below)) * KN;
            double x[XS];
            lds_block<XS>(xp, x);
#pragma unroll
            for (int m = 0; m < K; ++m) {
              double y[N];
              if ((N % 2 == 0)) lds_block<N>(yp + m * N, y);
              else {
#pragma unroll
                for (int c = 0; c < N; ++c) y[c] = yp[m * N + c];
              }
#pragma unroll
              for (int r = 0; r < M; ++r)
#pragma unroll
                for (int c = 0; c < N; ++c) acc[r * N + c] = fma(x[r * K + m], y[c], acc[r * N + c]);
            }
          }
        }
      }
      if (!PERSIST && slot >= 0) {
        if (EPI == 1) {
          // P(i,J) = P~(i,J) - omega * D_i^-1 * (A P~)(i,J)   (the block AXPY on the subset
          // pattern of PAPER.md:244 fused into the store of the product)
          const int64_t o = (int64_t)out + slot;
          const int32_t row = __ldg(a.out_row + o), own = __ldg(a.own_slot + o);
          const double* di = a.dinv + (int64_t)row * M * M;
          double z[MN];
#pragma unroll
          for (int r = 0; r < M; ++r)
#pragma unroll
            for (int c = 0; c < N; ++c) {
              double t = 0.0;
#pragma unroll
              for (int m = 0; m < M; ++m) t = fma(__ldg(di + r * M + m), acc[m * N + c], t);
              z[r * N + c] = t;
            }
#pragma unroll
          for (int e = 0; e < MN; ++e)
            acc[e] = fma(-a.omega, z[e], own >= 0 ? __ldg(a.own_vals + (int64_t)own * MN + e) : 0.0);
        }
        double* dst = a.cvals + (int64_t)(out + slot) * MN;
        if (MN % 2 == 0) {
#pragma unroll
          for (int e = 0; e < MN / 2; ++e) reinterpret_cast<double2*>(dst)[e] = make_double2(acc[2 * e], acc[2 * e + 1]);
        } else {
#pragma unroll
          for (int e = 0; e < MN; ++e) dst[e] = acc[e];
        }
      }
    }
    if (XBULK || YBULK) fence_async_smem();   // generic-proxy reads of this chunk before the next chunk's bulk writes
    __syncthreads();
  }
  if (PERSIST) {
    // partial blocks of the NW warps, added in warp order; every coarse block is written once
    double* part = reinterpret_cast<double*>(smem);
    if (lane < br_nslots) {
#pragma unroll
      for (int e = 0; e < MN; ++e) part[((int64_t)warp * br_nslots + lane) * MN + e] = acc[e];
    }
    __syncthreads();
    double* dst = a.cvals + (int64_t)bh.z * MN;
    for (int e = tid; e < br_nslots * MN; e += NT) {
      double v = part[e];
#pragma unroll
      for (int w = 1; w < NW; ++w) v += part[(int64_t)w * br_nslots * MN + e];
      dst[e] = v;
    }
  }
}

// prepare = true: the cold call (stream_upload) opts the kernel in to `smem` bytes of dynamic shared memory on the
// current device; false: the hot launch
template <int M, int K, int N>
static int stream_launch_mkn(const StreamArgs& a, bool persist, int64_t nbricks, int64_t smem, cudaStream_t st,
                             bool prepare) {
  if (persist) {
    auto kern = stream_product_kernel<M, K, N, STREAM_THREADS_PERSIST, true>;
    if (prepare) return optin_shared_memory(kern, smem);
    if (nbricks == 0) return BSR_OK;
    LAUNCH(kern, (unsigned)nbricks, STREAM_THREADS_PERSIST, (size_t)smem, st, a);
  } else {
    auto kern = stream_product_kernel<M, K, N, STREAM_THREADS_DIRECT, false>;
    if (prepare) return optin_shared_memory(kern, smem);
    if (nbricks == 0) return BSR_OK;
    LAUNCH(kern, (unsigned)nbricks, STREAM_THREADS_DIRECT, (size_t)smem, st, a);
  }
  return BSR_OK;
}

template <int M, int N>
static int stream_launch_smooth_mn(const StreamArgs& a, int64_t nbricks, int64_t smem, cudaStream_t st, bool prepare) {
  auto kern = stream_product_kernel<M, M, N, STREAM_THREADS_DIRECT, false, 1>;
  if (prepare) return optin_shared_memory(kern, smem);
  if (nbricks == 0) return BSR_OK;
  LAUNCH(kern, (unsigned)nbricks, STREAM_THREADS_DIRECT, (size_t)smem, st, a);
  return BSR_OK;
}

int stream_launch_smooth(int M, int N, const StreamArgs& a, int64_t nbricks, int64_t smem, cudaStream_t st,
                         bool prepare) {
  switch (M * 10 + N) {
    case 23: return stream_launch_smooth_mn<2, 3>(a, nbricks, smem, st, prepare);
    case 33: return stream_launch_smooth_mn<3, 3>(a, nbricks, smem, st, prepare);
    case 36: return stream_launch_smooth_mn<3, 6>(a, nbricks, smem, st, prepare);
    case 66: return stream_launch_smooth_mn<6, 6>(a, nbricks, smem, st, prepare);
  }
  return fail(BSR_ERR_BLOCK, "no staged smoothing kernel for <%d,%d,%d>", M, M, N);
}

int stream_launch(int M, int K, int N, const StreamArgs& a, bool persist, int64_t nbricks, int64_t smem, cudaStream_t st,
                  bool prepare) {
  const int key = M * 100 + K * 10 + N;
  switch (key) {
    case 222: return stream_launch_mkn<2, 2, 2>(a, persist, nbricks, smem, st, prepare);
    case 223: return stream_launch_mkn<2, 2, 3>(a, persist, nbricks, smem, st, prepare);
    case 323: return stream_launch_mkn<3, 2, 3>(a, persist, nbricks, smem, st, prepare);
    case 332: return stream_launch_mkn<3, 3, 2>(a, persist, nbricks, smem, st, prepare);
    case 232: return stream_launch_mkn<2, 3, 2>(a, persist, nbricks, smem, st, prepare);
    case 333: return stream_launch_mkn<3, 3, 3>(a, persist, nbricks, smem, st, prepare);
    case 336: return stream_launch_mkn<3, 3, 6>(a, persist, nbricks, smem, st, prepare);
    case 636: return stream_launch_mkn<6, 3, 6>(a, persist, nbricks, smem, st, prepare);
    case 663: return stream_launch_mkn<6, 6, 3>(a, persist, nbricks, smem, st, prepare);
    case 363: return stream_launch_mkn<3, 6, 3>(a, persist, nbricks, smem, st, prepare);
    case 666: return stream_launch_mkn<6, 6, 6>(a, persist, nbricks, smem, st, prepare);
  }
  return fail(BSR_ERR_BLOCK, "no staged product kernel for <%d,%d,%d>", M, K, N);
}

}  // namespace bsramg
