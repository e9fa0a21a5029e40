// ptap_prog.cu -- the hot kernels of ptap_numeric: brick-staged block products driven by lane programs
// (format and rationale: ptap_prog.h; host builder: ptap_prog.cpp).
//
// PAPER.md:219 (the dominant kernel is the numeric A*P with block sizes <3,3,6>), PAPER.md:103 ("local blocked triple
// product"), PAPER.md:97-99, 248-250 (coarse blocks summed through a precomputed block plan, contiguous bs_r*bs_c runs).
//
// One CTA = one brick.  Per chunk it (1) fetches the chunk's program words with one TMA bulk copy (cp.async.bulk,
// bytes counted on an mbarrier), (2) stages the X blocks (cp.async) and scatters the Y blocks to their class slots
// (coalesced 16-byte loads -> conflict-free 16-byte shared stores), (3) every lane walks its descriptor list: two
// shared-memory block loads and M*K*N fp64 FMAs per step, all 32 lanes busy, the quarter warps bank-conflict free on
// Y by construction.  Stage 1 writes each AP block once from registers (lists split over lanes are joined by a fixed
// shuffle tree first); stage 2 keeps one partial coarse block per lane over all chunks and adds the partial blocks of
// a coarse block in lane order through shared memory: the atomic-free segmented scatter into A_c.
#include "internal.h"
#include "ptap_prog.h"

namespace bsramg {

__device__ __forceinline__ int up16i(int b) { return (b + 15) & ~15; }

template <int BYTES>
__device__ __forceinline__ void cp_async(void* dst_smem, const void* src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(dst_smem);
  if (BYTES == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(src));
  else asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(src));
}
__device__ __forceinline__ void cp_async_wait_all() {
  asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count));
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
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

template <int NE>   // NE even, p 16-byte aligned
__device__ __forceinline__ void lds_block(const double* __restrict__ p, double (&v)[NE]) {
#pragma unroll
  for (int e = 0; e < NE / 2; ++e) {
    const double2 t = reinterpret_cast<const double2*>(p)[e];
    v[2 * e] = t.x;
    v[2 * e + 1] = t.y;
  }
}

template <int MN>
__device__ __forceinline__ void store_block(double* __restrict__ dst, const double (&acc)[MN]) {
  if (MN % 2 == 0) {
#pragma unroll
    for (int e = 0; e < MN / 2; ++e) reinterpret_cast<double2*>(dst)[e] = make_double2(acc[2 * e], acc[2 * e + 1]);
  } else {
#pragma unroll
    for (int e = 0; e < MN; ++e) dst[e] = acc[e];
  }
}

__device__ __forceinline__ void bulk_s2g(void* dst_global, const void* src_smem, unsigned bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
               ::"l"(dst_global), "r"((unsigned)__cvta_generic_to_shared(src_smem)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit_wait_read() {
  asm volatile("cp.async.bulk.commit_group;\n\tcp.async.bulk.wait_group.read 0;" ::: "memory");
}

__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }

// Persistent CTAs: CTA c works on bricks c, c + gridDim, ...  Shared memory: [record ring: 3][blob: 2][X][Y] ... and the
// output staging area at the very top, so that brick k+1 can be staged while the copy engine still reads brick k's
// rows.  Records are fetched two bricks ahead and blobs one chunk ahead (TMA bulk copies on mbarriers), so the only
// latency a brick waits for is that of its own operands, which are all in flight at once (cp.async).
template <int M, int K, int N, bool PERSIST>
__global__ void __launch_bounds__(PROG_NT, 3)
prog_kernel(const ProgArgs a) {
  constexpr int MK = M * K, KN = K * N, MN = M * N;
  constexpr int XS = (MK + 1) & ~1;                      // staged X block stride (doubles)
  constexpr int KNP = (KN + 1) & ~1;                     // doubles of a Y block read by a lane
  constexpr int YC16 = ((KNP / 2) & 1) ? KNP / 2 : KNP / 2 + 1;   // staged Y slot stride (16-byte units, odd)
  extern __shared__ __align__(16) unsigned char smem[];
  __shared__ uint64_t bar_rec[3], bar_blob[2];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nb = a.nbricks, stride = (int)gridDim.x;
  int b = (int)blockIdx.x;
  if (b >= nb) return;
  const int recb = a.rec_max_bytes, blobb = a.blob_max_bytes;
  unsigned char* blob_base = smem + 3 * recb;
  double* Xs = reinterpret_cast<double*>(blob_base + 2 * blobb);
  if (tid == 0) {
    mbar_init(&bar_rec[0], 1); mbar_init(&bar_rec[1], 1); mbar_init(&bar_rec[2], 1);
    mbar_init(&bar_blob[0], 1); mbar_init(&bar_blob[1], 1);
  }
  __syncthreads();
  auto fetch_rec = [&](int brick, int slot) {   // thread 0
    const int o0 = __ldg(a.rec_off + brick), o1 = __ldg(a.rec_off + brick + 1);
    mbar_arrive_expect_tx(&bar_rec[slot], (unsigned)(o1 - o0) * 4u);
    bulk_g2s(smem + slot * recb, a.rec + o0, (unsigned)(o1 - o0) * 4u, &bar_rec[slot]);
  };
  auto fetch_blob = [&](int at, int words, unsigned q) {   // thread 0
    mbar_arrive_expect_tx(&bar_blob[q & 1u], (unsigned)words * 4u);
    bulk_g2s(blob_base + (q & 1u) * blobb, a.blob + at, (unsigned)words * 4u, &bar_blob[q & 1u]);
  };
  unsigned q = 0;   // chunks processed so far by this CTA: blob buffer q & 1, phase (q >> 1) & 1
  if (tid == 0) {
    fetch_rec(b, 0);
    if (b + stride < nb) fetch_rec(b + stride, 1);
    mbar_wait(&bar_rec[0], 0u);
    const uint32_t* rec = reinterpret_cast<const uint32_t*>(smem);
    fetch_blob((int)rec[0], (int)rec[1], 0u);
  }
  bool stores_pending = false;   // this thread issued bulk stores whose shared-memory reads may still be in flight

  for (int it = 0; b < nb; b += stride, ++it) {
    const int rs = it % 3;
    mbar_wait(&bar_rec[rs], (unsigned)((it / 3) & 1));
    const uint32_t* rec = reinterpret_cast<const uint32_t*>(smem + rs * recb);
    const int nrows = (int)rec[2];
    const int32_t* tab = reinterpret_cast<const int32_t*>(rec + 4);   // xsrc[nrows], outbase[nrows], ysrc[nyrows]
    if (tid == 0 && b + 2 * stride < nb) fetch_rec(b + 2 * stride, (it + 2) % 3);   // ring slot of brick it-1: free
    double acc[MN];
#pragma unroll
    for (int e = 0; e < MN; ++e) acc[e] = 0.0;
    double* Cs = nullptr;
    const uint32_t* tables = nullptr;   // crow, fix, pstore of the program (behind the last chunk's program words)
    int nfix = 0;

    for (bool more = true; more; ++q) {
      mbar_wait(&bar_blob[q & 1u], (q >> 1) & 1u);
      const uint32_t* blob_s = reinterpret_cast<const uint32_t*>(blob_base + (q & 1u) * blobb);
      const int nx = (int)blob_s[PROG_H_NX], nyslots = (int)blob_s[PROG_H_NYSLOTS];
      const int nxrun = (int)blob_s[PROG_H_NXRUN], nycopy = (int)blob_s[PROG_H_NYCOPY];
      const unsigned wr01 = blob_s[PROG_H_ROUNDS01], wr23 = blob_s[PROG_H_ROUNDS23];
      const unsigned wl01 = blob_s[PROG_H_LEN01], wl23 = blob_s[PROG_H_LEN23];
      const int prog_words = (int)blob_s[PROG_H_PROG_WORDS];
      const int ncs = (int)blob_s[PROG_H_NCS], novf = (int)blob_s[PROG_H_NOVF];
      nfix = (int)blob_s[PROG_H_NFIX];
      const int next_blob = (int)blob_s[PROG_H_NEXT_BLOB], next_words = (int)blob_s[PROG_H_NEXT_WORDS];
      more = next_blob >= 0;
      if (tid == 0) {
        // the blob after this one: the next chunk of this brick, or the first chunk of the next brick (its record
        // was requested at least one brick ago).  Its buffer held the previous chunk, whose readers are done.
        if (more) fetch_blob(next_blob, next_words, q + 1u);
        else if (b + stride < nb) {
          mbar_wait(&bar_rec[(it + 1) % 3], (unsigned)(((it + 1) / 3) & 1));
          const uint32_t* nrec = reinterpret_cast<const uint32_t*>(smem + ((it + 1) % 3) * recb);
          fetch_blob((int)nrec[0], (int)nrec[1], q + 1u);
        }
      }
      auto rounds_of = [&](int w) { return (int)(((w < 2 ? wr01 : wr23) >> ((w & 1) * 16)) & 0xffffu); };
      auto len_of = [&](int w) { return (int)(((w < 2 ? wl01 : wl23) >> ((w & 1) * 16)) & 0xffffu); };
      const uint32_t* xruns = blob_s + PROG_H_WORDS;
      const uint32_t* ycp = xruns + 2 * nxrun;
      const uint32_t* prog = blob_s + ((PROG_H_WORDS + 2 * nxrun + nycopy + 3) & ~3);
      tables = prog + prog_words;
      unsigned char* Ys = reinterpret_cast<unsigned char*>(Xs) + up16i((nx + 8) * XS * 8);
      Cs = reinterpret_cast<double*>(smem + a.smem_total - up16i((ncs + novf) * MN * 8));
      // ---- operands: every copy is an asynchronous global -> shared copy, all in flight at once
      for (int r = warp; r < nxrun; r += PROG_NW) {
        const uint32_t w0 = xruns[2 * r], w1 = xruns[2 * r + 1];
        const int row = (int)(w0 & 0xffffu), k0 = (int)(w0 >> 16), n = (int)(w1 & 0xffffu), dstb = (int)(w1 >> 16);
        const double* src = a.xvals + ((int64_t)tab[row] + k0) * MK;
        double* dst = Xs + dstb * XS;
        if (MK % 2 == 0) {
          for (int c = lane; c < n * (MK / 2); c += 32) cp_async<16>(dst + 2 * c, src + 2 * c);
        } else {
          for (int e = lane; e < n * MK; e += 32) {
            const int blk = e / MK;
            cp_async<8>(dst + blk * XS + (e - blk * MK), src + e);
          }
        }
      }
      {
        constexpr int YB = (KN % 2 == 0) ? KN / 2 : KN;     // pieces per block (16-byte, or 8-byte for 3x3)
        constexpr int DB = PROG_NT / YB, DP = PROG_NT - DB * YB;   // a thread's next piece: block += DB, piece += DP
        const int npieces = nycopy * YB;
        const int32_t* ysrc = tab + 2 * nrows;
        int blk = tid / YB, pc = tid - blk * YB;
        for (int c = tid; c < npieces; c += PROG_NT) {
          const uint32_t yc = ycp[blk];                     // yrow | q << 12 | slot << 20
          const double* src = a.yvals + ((int64_t)ysrc[yc & 0xfffu] + (int)((yc >> 12) & 0xffu)) * KN;
          unsigned char* dst = Ys + (size_t)(yc >> 20) * (YC16 * 16);
          if (KN % 2 == 0) cp_async<16>(dst + pc * 16, src + 2 * pc);
          else cp_async<8>(dst + pc * 8, src + pc);
          blk += DB; pc += DP;
          if (pc >= YB) { pc -= YB; ++blk; }
        }
      }
      // the zero blocks padding steps multiply: X slots nx..nx+7 (eight bank groups) and Y slot c of every class c
      for (int e = tid; e < 8 * XS; e += PROG_NT) Xs[nx * XS + e] = 0.0;
      for (int e = tid; e < 8 * YC16 * 2; e += PROG_NT) reinterpret_cast<double*>(Ys)[e] = 0.0;
      cp_async_wait_all();
      if (stores_pending) { bulk_wait_read(); stores_pending = false; }   // the last brick's rows have left the staging area
      __syncthreads();
      // ---- this warp's program: rounds of G steps; a lane's list ends at the end of a round, where the lanes that
      // finished park their block in the staging area with one warp-wide store sequence
      {
        int doff = 0;
#pragma unroll
        for (int w = 0; w < PROG_NW; ++w)
          if (w < warp) doff += rounds_of(w) * (len_of(w) + (PERSIST ? 0 : 1)) * 32;
        const uint32_t* wd = prog + doff + lane;
        const int nr = rounds_of(warp), G = len_of(warp);
        for (int r = 0; r < nr; ++r) {
          uint32_t d = wd[0];
          for (int s = 0; s < G; ++s) {
            const uint32_t dn = wd[32 * (s + 1 < G ? s + 1 : s)];   // next descriptor: one latency off the chain
            const double* xp = Xs + (int)(d & 0xfffu) * XS;
            const double* yp = reinterpret_cast<const double*>(Ys + (size_t)((d >> 12) & 0xfffu) * (YC16 * 16));
            double x[XS], y[KNP];
            lds_block<XS>(xp, x);
            lds_block<KNP>(yp, y);
#pragma unroll
            for (int m = 0; m < K; ++m)
#pragma unroll
              for (int rr = 0; rr < M; ++rr)
#pragma unroll
                for (int c = 0; c < N; ++c) acc[rr * N + c] = fma(x[rr * K + m], y[m * N + c], acc[rr * N + c]);
            d = dn;
          }
          wd += 32 * G;
          if (!PERSIST) {
            const uint32_t sw = *wd;
            wd += 32;
            if (sw != PROG_NONE) {
              store_block<MN>(Cs + (size_t)sw * MN, acc);
#pragma unroll
              for (int e = 0; e < MN; ++e) acc[e] = 0.0;
            }
          }
        }
      }
      if (more) {
        fence_async_smem();   // this chunk's operands and blob were read through the generic proxy
        __syncthreads();
      }
    }
    __syncthreads();
    const uint32_t* crow = tables;
    const uint32_t* fix = crow + nrows;
    if (PERSIST) {
      // every lane parks its partial block: the first part of a coarse block in its output slot, the others in overflow
      const uint32_t ps = fix[2 * nfix + tid];
      if (ps != PROG_NONE) store_block<MN>(Cs + (size_t)ps * MN, acc);
      __syncthreads();
    }
    // ---- overflow parts are added to their block in a fixed order (no atomics), piece by piece
    {
      constexpr int P = (MN % 2 == 0) ? MN / 2 : MN;
      for (int e = tid; e < nfix * P; e += PROG_NT) {
        const int f = e / P, pc = e - f * P;
        const uint32_t h = fix[2 * f];
        const int cnt = (int)fix[2 * f + 1];
        const int main_slot = (int)(h & 0xffffu), first = (int)(h >> 16);
        if (MN % 2 == 0) {
          double2* mp = reinterpret_cast<double2*>(Cs + (size_t)main_slot * MN) + pc;
          double2 v = *mp;
          for (int k = 0; k < cnt; ++k) {
            const double2 t = reinterpret_cast<const double2*>(Cs + (size_t)(first + k) * MN)[pc];
            v.x += t.x; v.y += t.y;
          }
          *mp = v;
        } else {
          double v = Cs[(size_t)main_slot * MN + pc];
          for (int k = 0; k < cnt; ++k) v += Cs[(size_t)(first + k) * MN + pc];
          Cs[(size_t)main_slot * MN + pc] = v;
        }
      }
    }
    // ---- the brick's output rows leave shared memory: one TMA bulk store per row (contiguous bs_r*bs_c runs)
    if (MN % 2 == 0) {
      fence_async_smem();
      __syncthreads();
      for (int r = tid; r < nrows; r += PROG_NT) {
        const uint32_t cr = crow[r];
        const int cstart = (int)(cr & 0xffffu), len = (int)(cr >> 16);
        if (len > 0) {
          bulk_s2g(a.cvals + (int64_t)tab[nrows + r] * MN, Cs + (size_t)cstart * MN, (unsigned)len * MN * 8u);
          stores_pending = true;
        }
      }
      if (stores_pending) bulk_commit();
    } else {
      __syncthreads();
      for (int r = 0; r < nrows; ++r) {
        const uint32_t cr = crow[r];
        const int cstart = (int)(cr & 0xffffu), len = (int)(cr >> 16);
        double* dst = a.cvals + (int64_t)tab[nrows + r] * MN;
        for (int e = tid; e < len * MN; e += PROG_NT) dst[e] = Cs[(size_t)cstart * MN + e];
      }
    }
    fence_async_smem();   // record, blob and tables were read through the generic proxy; the copy engine writes them next
    __syncthreads();
  }
  if (stores_pending) bulk_wait_read();
}

template <int M, int K, int N, bool PERSIST>
static int launch_one(const ProgArgs& a, int64_t nbricks, int64_t smem, cudaStream_t st, bool prepare, int* ctas_per_sm) {
  auto kern = prog_kernel<M, K, N, PERSIST>;
  if (prepare) {   // cold: opt in to the device's full dynamic shared memory once per device context
    int dev = 0, optin = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    cudaFuncAttributes fa;
    CUDA_TRY(cudaFuncGetAttributes(&fa, kern));
    optin -= (int)fa.sharedSizeBytes;   // the kernel's static shared memory (the mbarrier) counts against the limit
    if (smem > optin) return fail(BSR_ERR_LIMIT, "a brick needs %lld bytes of shared memory, the device offers %d", (long long)smem, optin);
    CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, optin));
    if (ctas_per_sm) CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, kern, PROG_NT, (size_t)smem));
    return BSR_OK;
  }
  if (nbricks == 0) return BSR_OK;
  LAUNCH(kern, (unsigned)nbricks, PROG_NT, (size_t)smem, st, a);   // nbricks = persistent CTAs here (ProgDev::grid)
  return BSR_OK;
}

// prepare = true: cold call that sets the kernel's shared-memory attribute; false: the hot launch
int prog_launch(const ProgShape& sh, bool persist, const ProgArgs& a, int64_t nbricks, int64_t smem, cudaStream_t st,
                bool prepare, int* ctas_per_sm) {
  const int key = sh.M * 100 + sh.K * 10 + sh.N;
#define PK(m, k, n, p) return launch_one<m, k, n, p>(a, nbricks, smem, st, prepare, ctas_per_sm)
  if (!persist) {
    switch (key) {   // stage 1: <bf, bf, bc>
      case 222: PK(2, 2, 2, false);
      case 223: PK(2, 2, 3, false);
      case 332: PK(3, 3, 2, false);
      case 333: PK(3, 3, 3, false);
      case 336: PK(3, 3, 6, false);
      case 663: PK(6, 6, 3, false);
      case 666: PK(6, 6, 6, false);
    }
  } else {
    switch (key) {   // stage 2: <bc, bf, bc>
      case 222: PK(2, 2, 2, true);
      case 323: PK(3, 2, 3, true);
      case 232: PK(2, 3, 2, true);
      case 333: PK(3, 3, 3, true);
      case 636: PK(6, 3, 6, true);
      case 363: PK(3, 6, 3, true);
      case 666: PK(6, 6, 6, true);
    }
  }
#undef PK
  return fail(BSR_ERR_BLOCK, "no product kernel for <%d,%d,%d>", sh.M, sh.K, sh.N);
}

}  // namespace bsramg
