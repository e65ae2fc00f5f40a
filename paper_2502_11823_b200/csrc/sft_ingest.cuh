// sft_ingest.cuh - data SFTs from the time series on the GPU (section V.A:
// "SFTs can be computed online as data arrives", O(N0 log n_SFT)).  Computes Eq.(26) P:205,
//
//   x~_a[k] = dt sum_{j<n} x[a n + j] exp(-2 pi i j k / n),      k_lo <= k < k_hi,
//
// for every disjoint segment a of n = T_SFT fs samples (a trailing partial segment is dropped,
// DESIGN A13) and keeps ONLY the stored band: the time series is read from HBM exactly once (8 bytes per
// sample: this kernel's roofline) and (k_hi - k_lo) complex64 bins per SFT are written.
//
// n a power of two, 64 <= n <= 16384: one block per segment does a real-input FFT entirely in shared memory
// (227 KB per SM on B200: a 16384-sample segment packs into 8192 complex fp32 = 64 KB, three blocks per SM so
// that loads of one segment overlap the butterflies of another): z[j] = x[2j] + i x[2j+1], in-place radix-2
// decimation in frequency (output bit-reversed, read back through brev), twiddles from an fp64-evaluated table,
// then the split  X[k] = 1/2 [(Z[k] + conj Z[m-k]) - i w^k (Z[k] - conj Z[m-k])],  w = e^{-2 pi i / n}, for the band only.
// A band of at most 256 bins (n = 4096 ... 16384) takes sft_rfft_lowband_kernel: two radix-16 passes, then one short sum
// per wanted output instead of the remaining stages over all points.
// Any other n: direct summation over the band with exact integer phase reduction (j k mod n), fp64 accumulators.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sftk {

constexpr int FFT_MAX_N = 16384;

// twiddle table W[t] = exp(-2 pi i t / n), t < n/2 (fp64-evaluated, stored as complex64)
__global__ void sft_twiddle_kernel(int n, float2 *W) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n / 2) return;
  double s, c;
  sincospi(2.0 * (double)t / (double)n, &s, &c);
  W[t] = make_float2((float)c, (float)-s);
}

// Shared-memory index with one float2 of padding per 16: keeps every pass of the FFT bank-conflict free.
__device__ __forceinline__ int padi(int i) { return i + (i >> 4); }

__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
// v * exp(-2 pi i q / 16), q = 0..7 (compile-time after unrolling)
__device__ __forceinline__ float2 rot16(float2 v, int q) {
  const float c2 = 0.70710678118654752f, c1 = 0.92387953251128674f, s1 = 0.38268343236508977f;
  switch (q & 7) {
    case 0: return v;
    case 1: return make_float2(c1 * v.x + s1 * v.y, c1 * v.y - s1 * v.x);
    case 2: return make_float2(c2 * (v.x + v.y), c2 * (v.y - v.x));
    case 3: return make_float2(s1 * v.x + c1 * v.y, s1 * v.y - c1 * v.x);
    case 4: return make_float2(v.y, -v.x);
    case 5: return make_float2(c1 * v.y - s1 * v.x, -s1 * v.y - c1 * v.x);
    case 6: return make_float2(c2 * (v.y - v.x), -c2 * (v.x + v.y));
    default: return make_float2(s1 * v.y - c1 * v.x, -c1 * v.y - s1 * v.x);
  }
}

// R consecutive radix-2 DIF stages (half-blocks h, h/2, .., h >> (R-1)) on groups of 2^R points held in registers:
// the group of `base` is {base + j hl}, hl = h >> (R-1), j < 2^R; stage s couples j and j + 2^(R-1-s).  The twiddle of
// element j in stage s is exp(-2 pi i ((pos + j hl) mod hs) / 2 hs), hs = h >> s, i.e. w0^(2^s) times a multiple of a
// sixteenth of a turn, with w0 = exp(-2 pi i pos / 2h) the only table look-up of the group.  GLOBAL: the points come
// straight from the time series (z[j] = x[2j] + i x[2j+1], 16-byte loads) instead of shared memory (first pass).
template <int R, bool GLOBAL>
__device__ __forceinline__ void dif_pass(float2 *z, const double *seg, const float2 *W, int m, int n, int h, int tid, int nthr) {
  constexpr int G = 1 << R;
  const int hl = h >> (R - 1);
  const int tw = n / (2 * h);
  for (int g = tid; g < (m >> R); g += nthr) {
    const int pos = g & (hl - 1);
    const int base = ((g - pos) << R) + pos;          // groups tile blocks of 2h = hl * 2^R points
    float2 v[G];
#pragma unroll
    for (int j = 0; j < G; ++j) {
      if (GLOBAL) {
        const double2 d = __ldcs((const double2 *)seg + (base + j * hl));
        v[j] = make_float2((float)d.x, (float)d.y);
      } else {
        v[j] = z[padi(base + j * hl)];
      }
    }
    float2 wp = __ldg(W + pos * tw);                  // w0^(2^s)
#pragma unroll
    for (int s = 0; s < R; ++s) {
      const int hj = G >> (s + 1);                    // partner distance in j = points per half-block in units of hl
#pragma unroll
      for (int j = 0; j < G; ++j) {
        if ((j / hj) & 1) continue;
        const float2 u = v[j], w2 = v[j + hj];
        const float2 d = make_float2(u.x - w2.x, u.y - w2.y);
        v[j] = make_float2(u.x + w2.x, u.y + w2.y);
        // ((j hl) mod hs) / (2 hs) = (j mod hj) / (2 hj) of a turn = (j mod hj) * (8 / hj) sixteenths
        v[j + hj] = rot16(cmul(d, wp), (j % hj) * (8 / hj));
      }
      if (s + 1 < R) wp = cmul(wp, wp);
    }
#pragma unroll
    for (int j = 0; j < G; ++j) z[padi(base + j * hl)] = v[j];
  }
}

// Persistent blocks (grid = SMs x resident blocks), each walking the segments s = blockIdx.x, + gridDim.x, ...  While it works
// on a segment a block asks the TMA unit to pull its NEXT segment from HBM into L2 (cp.async.bulk.prefetch.L2), so that the
// first pass of that segment finds the samples in L2.  Dynamic shared memory: (n/2 + n/32 + 1) float2.
__global__ void __launch_bounds__(256) sft_rfft_band_kernel(const double *x, int n_sft, int n, int log2m, double dt, int k_lo, int nb,
                                                            const float2 *W, float2 *bins) {
  extern __shared__ float2 z[];
  const int m = n >> 1;
  for (int sidx = blockIdx.x; sidx < n_sft; sidx += gridDim.x) {
  const double *seg = x + (size_t)sidx * n;
  // next segment of this block -> L2, half after the first pass, half after the second (SFT_PF below the kernel explains why there)
  auto prefetch_half = [&](int half) {
    if (threadIdx.x == 0 && sidx + (int)gridDim.x < n_sft) {
      const double *nxt = x + (size_t)(sidx + gridDim.x) * n + half * (n / 2);
      asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(nxt), "r"((unsigned)(n * 4)) : "memory");
    }
  };
  int n_pf = 0;
  // in-place radix-2 DIF network over m points, up to four consecutive stages at a time in registers.  The first pass
  // reads the series from global memory (the only HBM traffic of the kernel) and leaves its output in shared memory.
  int h = m >> 1;                                    // half-block of the next stage
  int r = log2m;                                     // stages left
  dif_pass<4, true>(z, seg, W, m, n, h, threadIdx.x, blockDim.x);       // log2m >= 5
  h >>= 4; r -= 4;
  __syncthreads();
  prefetch_half(n_pf++);
  while (r >= 2) {
    if (r >= 4) { dif_pass<4, false>(z, seg, W, m, n, h, threadIdx.x, blockDim.x); h >>= 4; r -= 4; }
    else if (r == 3) { dif_pass<3, false>(z, seg, W, m, n, h, threadIdx.x, blockDim.x); h >>= 3; r -= 3; }
    else { dif_pass<2, false>(z, seg, W, m, n, h, threadIdx.x, blockDim.x); h >>= 2; r -= 2; }
    __syncthreads();
    if (n_pf < 2) prefetch_half(n_pf++);
  }
  if (n_pf < 2) prefetch_half(n_pf++);
  // r == 1: the last stage (pairs (2i, 2i+1), twiddle 1) is not run over the array: the few outputs needed below take
  // their butterfly themselves,  Z(pos) = z[pos] + z[pos+1] (pos even),  z[pos-1] - z[pos] (pos odd)
  const bool fold = r == 1;
  auto zout = [&](int pos) {
    const float2 v = z[padi(pos)];
    if (!fold) return v;
    const float2 w2 = z[padi(pos ^ 1)];
    return (pos & 1) ? make_float2(w2.x - v.x, w2.y - v.y) : make_float2(v.x + w2.x, v.y + w2.y);
  };
  // band bins from the bit-reversed m-point spectrum
  float2 *out = bins + (size_t)sidx * nb;
  const float fdt = (float)dt;
  for (int q = threadIdx.x; q < nb; q += blockDim.x) {
    const int k = k_lo + q;
    float2 X = make_float2(0.f, 0.f);
    if (k >= 0 && k <= m) {
      const int k1 = k & (m - 1), k2 = (m - k) & (m - 1);       // Z[m] = Z[0]
      const float2 A = zout((int)(__brev((unsigned)k1) >> (32 - log2m)));
      const float2 Bc = zout((int)(__brev((unsigned)k2) >> (32 - log2m)));
      const float2 B = make_float2(Bc.x, -Bc.y);                 // conj Z[m-k]
      const float2 S = make_float2(A.x + B.x, A.y + B.y), D = make_float2(A.x - B.x, A.y - B.y);
      float2 w;                                                  // w^k, k <= m = n/2
      if (k < m) w = __ldg(W + k); else w = make_float2(-1.f, 0.f);
      // -i w D = -i (wr + i wi)(Dr + i Di) = (wr Di + wi Dr) - i (wr Dr - wi Di)
      const float tr = w.x * D.y + w.y * D.x, ti = -(w.x * D.x - w.y * D.y);
      X = make_float2(0.5f * fdt * (S.x + tr), 0.5f * fdt * (S.y + ti));
    }
    out[q] = X;
  }
  __syncthreads();                                   // the work array is reused by the next segment
  }
}

// Second radix-16 pass of the narrow-band kernel below: groups {base + j B}, j < 16, of one 16 B-point block, pos = g mod B.
// Same network and output order as dif_pass<4, false> with h = 8 B, but the twiddle is applied once, after the four
// stages (which then contain sixteenth-turn rotations only): output j carries w^(pos bitrev4(j)), w = exp(-2 pi i / 16 B),
// read from the table tw[j][pos] in shared memory - pos = tid mod B is the same for every group a thread ever sees.
template <int LOG2B>
__device__ __forceinline__ void dif16_table_pass(float2 *z, const float2 *tw, int m, int tid, int nthr) {
  constexpr int B = 1 << LOG2B;
  const int pos = tid & (B - 1);
  for (int g = tid; g < (m >> 4); g += nthr) {
    const int base = ((g - pos) << 4) + pos;
    float2 v[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) v[j] = z[padi(base + j * B)];
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      const int hj = 8 >> s;
#pragma unroll
      for (int j = 0; j < 16; ++j) {
        if ((j / hj) & 1) continue;
        const float2 u = v[j], w2 = v[j + hj];
        v[j] = make_float2(u.x + w2.x, u.y + w2.y);
        v[j + hj] = rot16(make_float2(u.x - w2.x, u.y - w2.y), (j % hj) * (8 / hj));
      }
    }
    // z and tw are the same shared array to the compiler, so a twiddle load cannot move above an earlier store: the loads are
    // issued in batches of TWB ahead of their stores.  Measured (ms): TWB = 1 0.2880, 2 0.2838, 3 0.2850, 4 0.2875, 8 0.2893,
    // all fifteen 0.3316 (spills at the 80-register cap).
    constexpr int TWB = 2;
    z[padi(base)] = v[0];
#pragma unroll
    for (int j0 = 1; j0 < 16; j0 += TWB) {
      float2 t[TWB];
#pragma unroll
      for (int i = 0; i < TWB; ++i) if (j0 + i < 16) t[i] = tw[(j0 + i) * B + pos];
#pragma unroll
      for (int i = 0; i < TWB; ++i) if (j0 + i < 16) z[padi(base + (j0 + i) * B)] = cmul(v[j0 + i], t[i]);
    }
  }
}

// Narrow band (at most 256 bins, 1 <= k_lo, k_hi <= m = n/2): output-pruned version of the kernel above.  After the first eight
// DIF stages (two radix-16 passes) the work array is 256 independent blocks of B = m/256 points: block b holds the sub-problem
// of the outputs k = r + 256 k'', r = bitrev8(b), and  Z[k] = sum_{j<B} y_b[j] exp(-2 pi i j k''/B).  A band of <= 256 bins
// meets every residue r at most once, and so does its mirror image m - k (needed by the real-input split): instead of running
// the remaining log2(B) stages over all m points, thread b sums its block once for each of the (at most two) outputs asked of
// it - 2 B complex multiply-adds per thread against the third radix-16 pass, the last radix-2 stage and the bit-reversed
// gather.  Twiddles of the four values k'' can take come from a table in shared memory (T, filled once per block); the
// k'' = 0 sums of a band below bin 256 need none.  blockDim.x == 256.  Dynamic shared memory: (n/2 + n/32 + 1 + 20 B) float2.
// Asks the TMA unit to pull `bytes_` bytes at double offset `off_` of this block's NEXT segment from HBM into L2
// (cp.async.bulk.prefetch.L2, one instruction, SASS UBLKPF).  Issued in the phases that do not read global memory - half a
// segment after the first pass, half after the second - so that the HBM reads run under the shared-memory passes instead of
// beside the block's own loads: 0.317 -> 0.289 ms against one prefetch at the top of the segment (0.349 without).
// (All resident blocks together hold <= 444 x 128 KB = 57 MB of prefetched segments, under half of B200's L2.)
#define SFT_PF(off_, bytes_) do { if (threadIdx.x == 0 && sidx + pf_stride < n_sft) { \
    const double *nxt_ = x + (size_t)(sidx + pf_stride) * n + (off_); \
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(nxt_), "r"((unsigned)(bytes_)) : "memory"); } } while (0)
template <int LOG2B>
__global__ void __launch_bounds__(256, 3) sft_rfft_lowband_kernel(const double *x, int n_sft, double dt, int k_lo, int nb,
                                                               const float2 *W, float2 *bins, int pf_stride) {
  constexpr int B = 1 << LOG2B, m = 256 << LOG2B, n = 2 * m;       // compile-time sizes: every shared-memory offset folds
  extern __shared__ float2 z[];
  const int k_hi = k_lo + nb;
  float2 *T = z + (m + (m >> 4) + 1);                   // [4][B]: slots {a0, a0 + 1, c0, c0 + 1}
  float2 *T2 = T + 4 * B;                               // [16][B]: twiddles of the second pass (dif16_table_pass)
  for (int t = threadIdx.x; t < 16 * B; t += blockDim.x) {
    const int j = t >> LOG2B, pos = t & (B - 1);
    const int q = (int)(__brev((unsigned)j) >> 28);     // exp(-2 pi i pos q / 16 B) = W[pos q n / 16 B], pos q < 16 B / 2 ... 16 B
    const int e = pos * q;                              // < 16 B
    const float2 w = __ldg(W + (e & (8 * B - 1)) * (n >> (LOG2B + 4)));
    T2[t] = (e & (8 * B)) ? make_float2(-w.x, -w.y) : w;
  }
  const int a0 = k_lo >> 8, c0 = (m - k_hi + 1) >> 8;
  for (int t = threadIdx.x; t < 4 * B; t += blockDim.x) {
    const int slot = t >> LOG2B, j = t & (B - 1);
    const int kpp = ((slot < 2 ? a0 : c0) + (slot & 1)) & (B - 1);
    const int e = (j * kpp) & (B - 1);                  // exp(-2 pi i e / B) = +- W[(e mod B/2) n/B]
    const float2 w = __ldg(W + (e & (B / 2 - 1)) * (n >> LOG2B));
    T[t] = (e & (B / 2)) ? make_float2(-w.x, -w.y) : w;
  }
  // the outputs asked of this thread's block (the same for every segment)
  // Block b of this thread: for B >= 16 one of the 32 blocks that its own warp writes in the second pass (B = 32: warp w
  // transforms the 512-point chunks w and w + 8 = blocks 16 w .. 16 w + 15 and 16 (w + 8) ..; B = 16: chunks 2 w, 2 w + 1 =
  // blocks 32 w .. 32 w + 31), so that the sums need a __syncwarp() after that pass, not a block-wide barrier.
  constexpr bool WARP_LOCAL = LOG2B >= 4;
  const int lane_ = threadIdx.x & 31, warp_ = threadIdx.x >> 5;
  const int b = LOG2B == 5 ? 16 * (warp_ + 8 * (lane_ >> 4)) + (lane_ & 15) : (int)threadIdx.x;
  const int r = (int)(__brev((unsigned)b) >> 24);
  const int kA = k_lo + ((r - k_lo) & 255), kM = k_lo + ((-r - k_lo) & 255);       // band bins with k = r, m - k = r (mod 256)
  const bool hasA = kA < k_hi, hasM = kM < k_hi;
  const float2 *TA = T + (((kA >> 8) - a0) & 1) * B, *TM = T + (2 + ((((m - kM) >> 8) - c0) & 1)) * B;
  const bool plainA = k_hi <= 256;                      // every k'' of the band itself is 0
  const float2 *blk = z + (b * B + ((b * B) >> 4));
  const float fdt = (float)dt;
  __syncthreads();
  // Results: slot p = q ^ (q >> 4) for band offset q (the threads of a warp hold residues that differ in their high bits
  // only), the mirror sums 256 slots further.  With m/16 >= 512 the slots are the padding entries of the work array (index
  // 17 p + 16), which no pass ever touches, and the read-out of segment s (split + store of the band) is deferred to just
  // after the first barrier of the block's next segment, which already orders it after every thread's result write.  The
  // opposite order - no thread may overwrite the slots before every thread has read them - is kept by an mbarrier on which
  // all threads arrive after their read-out and wait before their next result write; that wait is over long before it is
  // reached (a second pass and the block sums lie in between).  One block-wide barrier per segment is left, after the first
  // pass (five before: 0.283 -> 0.266 ms).  Smaller transforms keep the results in the first 512 entries, between barriers.
  constexpr bool PADRES = m / 16 >= 512;
  __shared__ unsigned long long bar_mem;
  const unsigned bar_s = (unsigned)__cvta_generic_to_shared(&bar_mem);
  if (PADRES && threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared.b64 [%0], %1;" ::"r"(bar_s), "r"(256) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  auto slot = [](int p) { return PADRES ? 17 * p + 16 : p; };
  auto read_out = [&](int sdone) {
    float2 *out = bins + (size_t)sdone * nb;
    for (int q = threadIdx.x; q < nb; q += blockDim.x) {
      const int k = k_lo + q;
      const float2 A = z[slot(q ^ (q >> 4))], Bc = z[slot(256 + (q ^ (q >> 4)))];
      const float2 Bv = make_float2(Bc.x, -Bc.y);                 // conj Z[m-k]
      const float2 S = make_float2(A.x + Bv.x, A.y + Bv.y), D = make_float2(A.x - Bv.x, A.y - Bv.y);
      float2 w;                                                  // w^k, k <= m = n/2
      if (k < m) w = __ldg(W + k); else w = make_float2(-1.f, 0.f);
      const float tr = w.x * D.y + w.y * D.x, ti = -(w.x * D.x - w.y * D.y);
      out[q] = make_float2(0.5f * fdt * (S.x + tr), 0.5f * fdt * (S.y + ti));
    }
  };
  int pending = -1;                                    // PADRES: segment whose results wait in the padding entries
  unsigned phase = 0;                                  // parity of the mbarrier phase to wait for
  for (int sidx = blockIdx.x; sidx < n_sft; sidx += gridDim.x) {
    const double *seg = x + (size_t)sidx * n;
    dif_pass<4, true>(z, seg, W, m, n, m >> 1, threadIdx.x, blockDim.x);
    __syncthreads();
    SFT_PF(0, n * 4);                                  // first half of this block's next segment -> L2 (see SFT_PF)
    if (PADRES) {
      // read-out of the block's previous segment: this barrier already orders it after every thread's result write
      if (pending >= 0) read_out(pending);
      asm volatile("{ .reg .b64 t; mbarrier.arrive.shared.b64 t, [%0]; }" ::"r"(bar_s) : "memory");   // "I have read the results"
    }
    dif16_table_pass<LOG2B>(z, T2, m, threadIdx.x, blockDim.x);
    if (WARP_LOCAL) __syncwarp(); else __syncthreads();
    SFT_PF(n / 2, n * 4);                              // second half
    float2 sA = make_float2(0.f, 0.f), sM = sA;
#pragma unroll
    for (int j = 0; j < B; ++j) {
      const float2 v = blk[j + (j >> 4)];
      if (plainA) {
        sA.x += v.x; sA.y += v.y;
      } else {
        const float2 t = TA[j];
        sA.x = fmaf(v.x, t.x, fmaf(-v.y, t.y, sA.x)); sA.y = fmaf(v.x, t.y, fmaf(v.y, t.x, sA.y));
      }
      const float2 u = TM[j];
      sM.x = fmaf(v.x, u.x, fmaf(-v.y, u.y, sM.x)); sM.y = fmaf(v.x, u.y, fmaf(v.y, u.x, sM.y));
    }
    if (!PADRES) __syncthreads();                      // every block has been read: the array now takes the results
    if (PADRES) {                                      // every thread has read the previous results (long ago, as a rule)
      unsigned ok;
      do {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(ok) : "r"(bar_s), "r"(phase) : "memory");
      } while (!ok);
      phase ^= 1u;
    }
    if (hasA) z[slot((kA - k_lo) ^ ((kA - k_lo) >> 4))] = sA;                 // Z[k]
    if (hasM) z[slot(256 + ((kM - k_lo) ^ ((kM - k_lo) >> 4)))] = sM;         // Z[m - k]
    if (PADRES) {
      pending = sidx;
    } else {
      __syncthreads();
      read_out(sidx);
      __syncthreads();                                 // the work array is reused by the next segment
    }
  }
  if (PADRES && pending >= 0) {
    __syncthreads();
    read_out(pending);
  }
}

// Direct band DFT for any n: block per segment, one thread per bin, samples staged through shared memory.
__global__ void __launch_bounds__(256) sft_dft_band_kernel(const double *x, int n, double dt, int k_lo, int nb, float2 *bins) {
  __shared__ double xs[1024];
  const double *seg = x + (size_t)blockIdx.x * n;
  for (int q0 = 0; q0 < nb; q0 += blockDim.x) {
    const int q = q0 + threadIdx.x, k = k_lo + q;
    double re = 0.0, im = 0.0;
    long long ph = 0;                                 // (j k) mod n, exact
    const long long kk = ((long long)k % n + n) % n;
    for (int j0 = 0; j0 < n; j0 += 1024) {
      __syncthreads();
      for (int j = threadIdx.x; j < 1024 && j0 + j < n; j += blockDim.x) xs[j] = seg[j0 + j];
      __syncthreads();
      const int je = min(1024, n - j0);
      if (q < nb) {
        for (int j = 0; j < je; ++j) {
          double s, c;
          sincospi(2.0 * (double)ph / (double)n, &s, &c);
          re = fma(xs[j], c, re);
          im = fma(xs[j], -s, im);
          ph += kk;
          if (ph >= n) ph -= n;
        }
      }
    }
    if (q < nb) bins[(size_t)blockIdx.x * nb + q] = make_float2((float)(dt * re), (float)(dt * im));
  }
}

// ---------------------------------------------------------------------------------------------
// Per-SFT noise level from the data themselves ("whitening data on a per-SFT basis").  With the
// separable noise model S_a(f_k) = s_a S(f_k) (DESIGN A9) and Gaussian noise, |x~_{a,k}|^2 / (S(f_k) T/2) is s_a times a unit
// exponential variate, whose median is ln 2:
//   s^_a = median{ |x~_{a',k}|^2 / (S(f_k) T/2) : |a' - a| <= w, a' not a gap, k valid } / ln 2.
// The median over the band (and over 2w+1 neighbouring SFTs) is insensitive to a narrow-band signal crossing it.  An SFT whose
// bins are all exactly zero is a gap (s^ = 0) and does not enter its neighbours' pools.
constexpr int PSD_MAX_VALUES = 8192;

__global__ void sft_nonzero_kernel(const float2 *bins, int nb, unsigned char *flag) {
  __shared__ int any;
  if (threadIdx.x == 0) any = 0;
  __syncthreads();
  const float2 *row = bins + (size_t)blockIdx.x * nb;
  int a = 0;
  for (int q = threadIdx.x; q < nb; q += blockDim.x) a |= (row[q].x != 0.f) | (row[q].y != 0.f);
  if (a) any = 1;
  __syncthreads();
  if (threadIdx.x == 0) flag[blockIdx.x] = (unsigned char)any;
}

// One block per SFT; npow2 = the power of two >= the largest pool size (<= PSD_MAX_VALUES); bitonic sort in shared memory.
__global__ void __launch_bounds__(256) sft_psd_scale_kernel(const float2 *bins, const unsigned char *flag, const double *shape,
                                                            int n_sft, int nb, int k_lo, int n_samp, double half_T, int w, int npow2,
                                                            double *scale) {
  extern __shared__ float vals[];
  __shared__ int count;
  const int a = blockIdx.x;
  if (!flag[a]) {
    if (threadIdx.x == 0) scale[a] = 0.0;
    return;
  }
  if (threadIdx.x == 0) count = 0;
  __syncthreads();
  const int q0 = max(0, 1 - k_lo), q1 = min(nb, n_samp / 2 - k_lo);        // valid bins 1 <= k <= n/2 - 1
  const int nv = max(0, q1 - q0);
  int slot = 0;                                                            // pool layout: [present neighbour][valid bin]
  for (int b = max(0, a - w); b <= min(n_sft - 1, a + w); ++b) {
    if (!flag[b]) continue;
    const float2 *row = bins + (size_t)b * nb;
    for (int q = threadIdx.x; q < nv; q += blockDim.x) {
      const float2 v = row[q0 + q];
      const double Sk = shape ? shape[q0 + q] : 1.0;
      vals[slot * nv + q] = (float)(((double)v.x * (double)v.x + (double)v.y * (double)v.y) / (Sk * half_T));
    }
    ++slot;
  }
  const int cnt = slot * nv;
  for (int i = cnt + threadIdx.x; i < npow2; i += blockDim.x) vals[i] = __int_as_float(0x7f800000);   // +inf padding
  __syncthreads();
  for (int k = 2; k <= npow2; k <<= 1) {
    for (int j = k >> 1; j > 0; j >>= 1) {
      for (int i = threadIdx.x; i < npow2; i += blockDim.x) {
        const int l = i ^ j;
        if (l > i) {
          const float x = vals[i], y = vals[l];
          const bool up = (i & k) == 0;
          if ((x > y) == up) { vals[i] = y; vals[l] = x; }
        }
      }
      __syncthreads();
    }
  }
  if (threadIdx.x == 0) {
    double med = 0.0;
    if (cnt > 0) med = (cnt & 1) ? (double)vals[cnt / 2] : 0.5 * ((double)vals[cnt / 2 - 1] + (double)vals[cnt / 2]);
    scale[a] = med / 0.6931471805599453;
  }
}

}  // namespace sftk
