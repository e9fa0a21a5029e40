// ptap_stream.cu -- the hot kernels of ptap_numeric: brick-staged, output-stationary block products.
//
// PAPER.md:219 (the dominant kernel is the numeric A*P with block sizes <3,3,6>), PAPER.md:103 ("local blocked triple
// product"), PAPER.md:97-99, 248-250 (coarse blocks summed through a precomputed block plan, contiguous bs_r*bs_c
// runs).  Schedule format: internal.h / ptap_stream.cpp.
//
// One CTA = one brick.  Per chunk it stages, with coalesced loads, the X blocks (A rows / a piece of an R row), every
// Y row they reference (P rows / AP rows), the product codes and the item table in shared memory.  Then lane groups
// of N lanes (lane = column c of the output block) walk their items: per product a group reads its X block by
// broadcast (M*K doubles, 16-byte loads) and column c of the Y block (K doubles), and keeps the M x N output block in
// M registers per lane.  HBM sees each operand once per brick (Y again from L2 for neighbouring bricks); the
// gathers that made the one-thread-per-block version L1-bound (profiles/r1a_first_path.md) are shared-memory reads.
// No atomics: a block is either written once from registers (stage 1) or its parts are added in plan order into the
// brick's shared-memory accumulator and written once (stage 2).
#include "internal.h"
#include "ptap_stream.h"

namespace bsramg {

__device__ __forceinline__ int64_t up16d(int64_t b) { return (b + 15) & ~int64_t(15); }

template <int M, int K, int N, typename CodeT, int OXBITS>
__global__ void __launch_bounds__(STREAM_THREADS, 2)
stream_product_kernel(const StreamArgs a) {
  constexpr int MK = M * K, KN = K * N, MN = M * N, XS = (MK + 1) & ~1;
  constexpr int G = 32 / N;                      // lane groups per warp
  constexpr int NG = (STREAM_THREADS / 32) * G;  // lane groups per CTA
  extern __shared__ __align__(16) unsigned char smem[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int b = blockIdx.x;
  const int g = lane / N, c = lane % N;
  const bool glive = g < G;
  const int gid = warp * G + g;

  const int acc0 = a.br_acc_ptr[b], nacc = a.br_acc_ptr[b + 1] - acc0;
  double* accs = reinterpret_cast<double*>(smem);
  unsigned char* chunk_base = smem + up16d((int64_t)nacc * MN * 8);
  for (int e = tid; e < nacc * MN; e += STREAM_THREADS) accs[e] = 0.0;

  for (int ch = a.br_chunk_ptr[b]; ch < a.br_chunk_ptr[b + 1]; ++ch) {
    const int nx = a.ch_nx[ch], ny = a.ch_ny[ch], nparts = a.ch_nparts[ch];
    const int item0 = a.ch_item_ptr[ch], nitems = a.ch_item_ptr[ch + 1] - item0;
    const int64_t code0 = a.ch_code_ptr[ch];
    const int ncodes = (int)(a.ch_code_ptr[ch + 1] - code0);
    double* Xs = reinterpret_cast<double*>(chunk_base);
    double* Ys = reinterpret_cast<double*>(chunk_base + up16d((int64_t)nx * XS * 8));
    double* parts = Ys + (up16d((int64_t)ny * KN * 8) >> 3);
    CodeT* codes = reinterpret_cast<CodeT*>(reinterpret_cast<unsigned char*>(parts) + up16d((int64_t)nparts * MN * 8));
    int32_t* items = reinterpret_cast<int32_t*>(reinterpret_cast<unsigned char*>(codes) + up16d((int64_t)ncodes * sizeof(CodeT)));
    int32_t* gptr = items + (up16d((int64_t)nitems * 12) >> 2);
    // ---- stage X (padded to XS doubles per block), Y, codes, items, group pointers
    for (int r = a.ch_xrun_ptr[ch]; r < a.ch_xrun_ptr[ch + 1]; ++r) {
      const StreamRun run = a.xruns[r];
      if (MK % 2 == 0) {
        const double2* src = reinterpret_cast<const double2*>(a.xvals + (int64_t)run.src * MK);
        double2* dst = reinterpret_cast<double2*>(Xs + (int64_t)run.dst * XS);
        for (int e = tid; e < run.n * (MK / 2); e += STREAM_THREADS) dst[e] = __ldcs(src + e);
      } else {
        const double* src = a.xvals + (int64_t)run.src * MK;
        double* dst = Xs + (int64_t)run.dst * XS;
        for (int e = tid; e < run.n * MK; e += STREAM_THREADS) {
          const int blk = e / MK;
          dst[blk * XS + (e - blk * MK)] = __ldcs(src + e);
        }
      }
    }
    for (int r = a.ch_yrun_ptr[ch]; r < a.ch_yrun_ptr[ch + 1]; ++r) {
      const StreamRun run = a.yruns[r];
      if (KN % 2 == 0) {
        const double2* src = reinterpret_cast<const double2*>(a.yvals + (int64_t)run.src * KN);
        double2* dst = reinterpret_cast<double2*>(Ys + (int64_t)run.dst * KN);
        for (int e = tid; e < run.n * (KN / 2); e += STREAM_THREADS) dst[e] = __ldg(src + e);
      } else {
        const double* src = a.yvals + (int64_t)run.src * KN;
        double* dst = Ys + (int64_t)run.dst * KN;
        for (int e = tid; e < run.n * KN; e += STREAM_THREADS) dst[e] = __ldg(src + e);
      }
    }
    {
      const CodeT* src = reinterpret_cast<const CodeT*>(a.codes) + code0;
      for (int e = tid; e < ncodes; e += STREAM_THREADS) codes[e] = __ldcs(src + e);
      const int32_t* isrc = reinterpret_cast<const int32_t*>(a.items + item0);
      for (int e = tid; e < nitems * 3; e += STREAM_THREADS) items[e] = __ldcs(isrc + e);
      const int32_t* gsrc = a.ch_gptr + (int64_t)ch * (NG + 1);
      for (int e = tid; e <= NG; e += STREAM_THREADS) gptr[e] = __ldcs(gsrc + e);
    }
    __syncthreads();
    // ---- the product streams
    {
      int it = glive ? gptr[gid] : 0;
      const int it_end = glive ? gptr[gid + 1] : 0;
      int rem = 0, out = 0, xb = 0;
      const CodeT* cp = codes;
      double acc[M];
#pragma unroll
      for (int r = 0; r < M; ++r) acc[r] = 0.0;
      while (true) {
        const bool have = rem > 0 || it < it_end;
        if (!__any_sync(0xffffffffu, have)) break;
        if (have) {
          if (rem == 0) {
            out = items[3 * it];
            cp = codes + items[3 * it + 1];
            const uint32_t w = (uint32_t)items[3 * it + 2];
            rem = (int)(w & 0xffffu);
            xb = (int)(w >> 16);
            ++it;
#pragma unroll
            for (int r = 0; r < M; ++r) acc[r] = 0.0;
          }
          const uint32_t code = (uint32_t)(*cp++);
          const double* xp = Xs + (xb + (int)(code & ((1u << OXBITS) - 1u))) * XS;
          const double* yp = Ys + (int)(code >> OXBITS) * KN + c;
          double y[K], x[XS];
#pragma unroll
          for (int m = 0; m < K; ++m) y[m] = yp[m * N];
#pragma unroll
          for (int e = 0; e < XS / 2; ++e) {
            const double2 t = reinterpret_cast<const double2*>(xp)[e];
            x[2 * e] = t.x;
            x[2 * e + 1] = t.y;
          }
#pragma unroll
          for (int r = 0; r < M; ++r)
#pragma unroll
            for (int m = 0; m < K; ++m) acc[r] = fma(x[r * K + m], y[m], acc[r]);
          if (--rem == 0) {
            double* dst = (out >= 0) ? a.cvals + (int64_t)out * MN + c : parts + (-out - 1) * MN + c;
#pragma unroll
            for (int r = 0; r < M; ++r) dst[r * N] = acc[r];
          }
        }
      }
    }
    __syncthreads();
    // ---- parts -> brick accumulator, in plan order
    {
      const int red0 = a.ch_red_ptr[ch], nred = a.ch_red_ptr[ch + 1] - red0;
      for (int e = tid; e < nred * MN; e += STREAM_THREADS) {
        const int ri = e / MN, el = e - ri * MN;
        const StreamRed rd = a.reds[red0 + ri];
        double v = accs[rd.acc * MN + el];
        for (int q = 0; q < rd.nparts; ++q) v += parts[(rd.part0 + q) * MN + el];
        accs[rd.acc * MN + el] = v;
      }
    }
    __syncthreads();
  }
  // ---- the brick's accumulated blocks, written once
  for (int e = tid; e < nacc * MN; e += STREAM_THREADS) {
    const int ai = e / MN, el = e - ai * MN;
    a.cvals[(int64_t)a.acc_slot[acc0 + ai] * MN + el] = accs[e];
  }
}

template <int M, int K, int N>
static int stream_launch_mkn(const StreamArgs& a, bool wide, int64_t nbricks, int64_t smem, cudaStream_t st) {
  if (nbricks == 0) return BSR_OK;
  if (wide) {
    auto kern = stream_product_kernel<M, K, N, uint32_t, 12>;
    static int64_t set_smem = -1;
    if (smem > set_smem) {
      CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      set_smem = smem;
    }
    LAUNCH(kern, (unsigned)nbricks, STREAM_THREADS, (size_t)smem, st, a);
  } else {
    auto kern = stream_product_kernel<M, K, N, uint16_t, 5>;
    static int64_t set_smem = -1;
    if (smem > set_smem) {
      CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      set_smem = smem;
    }
    LAUNCH(kern, (unsigned)nbricks, STREAM_THREADS, (size_t)smem, st, a);
  }
  return BSR_OK;
}

int stream_launch(int M, int K, int N, const StreamArgs& a, bool wide, int64_t nbricks, int64_t smem, cudaStream_t st) {
  const int key = M * 100 + K * 10 + N;
  switch (key) {
    case 222: return stream_launch_mkn<2, 2, 2>(a, wide, nbricks, smem, st);
    case 223: return stream_launch_mkn<2, 2, 3>(a, wide, nbricks, smem, st);
    case 323: return stream_launch_mkn<3, 2, 3>(a, wide, nbricks, smem, st);
    case 332: return stream_launch_mkn<3, 3, 2>(a, wide, nbricks, smem, st);
    case 232: return stream_launch_mkn<2, 3, 2>(a, wide, nbricks, smem, st);
    case 333: return stream_launch_mkn<3, 3, 3>(a, wide, nbricks, smem, st);
    case 336: return stream_launch_mkn<3, 3, 6>(a, wide, nbricks, smem, st);
    case 636: return stream_launch_mkn<6, 3, 6>(a, wide, nbricks, smem, st);
    case 663: return stream_launch_mkn<6, 6, 3>(a, wide, nbricks, smem, st);
    case 363: return stream_launch_mkn<3, 6, 3>(a, wide, nbricks, smem, st);
    case 666: return stream_launch_mkn<6, 6, 6>(a, wide, nbricks, smem, st);
  }
  return fail(BSR_ERR_BLOCK, "no stream kernel for <%d,%d,%d>", M, K, N);
}

int stream_groups(int N) { return (STREAM_THREADS / 32) * (32 / N); }

}  // namespace bsramg
