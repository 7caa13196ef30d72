// gm_tc.cuh -- SURVEY 8(f)-4: the PSF convolution on the 5th-generation tensor cores
// (tcgen05.mma, accumulators and the image operand in tensor memory), as a stand-alone
// engine behind gm_conv (include/gm.h), judged against the same oracle as the FFMA2 loop.
//
// Formulation.  M[i,j] = sum_{a,b} P[a,b] S[i+a-h, j+b-h] (P = the flipped PSF, R:C1).  The image
// is cut into TILES of kTileR x kTileC = 4 rows x 32 columns; tile m of a 128 x 128 cutout is LANE m
// of the tensor memory (128 lanes = the M dimension of one MMA).  For window row y (0 .. kTileR+K-2) of
// every tile at once and output row r of the tile, tap row a = y - r contributes
//
//     D_r[m, j] += sum_c  A_y[m, c] * T_a[c, j],   T_a[c, j] = P[a, c - j]   (a Toeplitz band),
//
// an MMA of shape 128 x 32 x 16 per 16 window columns c: A_y[m, :] = the window row of tile m
// (tensor memory, written by the producer warps), T_a = 16 x 32 band blocks in shared memory,
// D_r = 32 fp32 columns of tensor memory.  T_a[c0 + r', j] depends on (r' - (j - c0)) only, so all
// chunks c0 of a tap row are 32-row windows of ONE 16-column matrix E_a stored once per tap row
// (canonical K-major no-swizzle layout, 16-byte rows: a window is just a start address).
//
// Tile shape (measured, profiles/r02_tc_engine.md).  The band wastes (N + K - 1) / K of the tensor work, so a
// narrower tile looks better on paper, and the code builds with 8 x 16 tiles (N = 16, the smallest N of an
// M = 128 MMA).  On the B200 a 128 x 16 x 16 MMA takes ~13 cycles, not the 8 its size suggests (128 x 32 x 16:
// 16.0), so the 1.5x more MMAs of N = 16 made every configuration slower (C1 50 -> 58 ms, P1 682 -> 883 ms),
// and the 8-row tile leaves up to 7 tap rows after an accumulator's centre row, which triples the truncation
// bias of the accumulator (below).  4 x 32 stays.
//
// Precision.  fp32 operands are split into two fp16 halves after an exact power-of-two scaling
// per image and per PSF, x = hi + lo with hi = fp16(x), lo = fp16(x - hi) (22 significant
// bits), and three MMAs accumulate hi*hi + lo*hi + hi*lo in fp32; the lo*lo term (2^-22
// relative) is dropped.  fp16 runs at twice the TF32 rate with K = 16 per instruction, so this
// costs 1.5 TF32-equivalents per product instead of 3.
//
// Pipeline of one CTA (one per SM, persistent over galaxies), all hand-offs by mbarrier:
//   warps 4-7   load cutout g+1 (global fp32 -> shared (hi, lo) fp16 pairs, one word per
//               pixel), then drain the accumulators of cutout g (tcgen05.ld -> global)
//   warps 0-3   window row y of every tile: LDS.128 -> PRMT -> tcgen05.st (3 row buffers)
//   warps 8-11  issue the MMAs (converged warp, one elected lane), one accumulator row each
//   warp 12     streams the E_a of the tap rows into two rings with cp.async.bulk (TMA)
// Measured issue rates (B200): one converged warp issues a 128 x 32 x 16 MMA every 16.0 clk, the tensor-core
// floor for that shape; four warps issue, one accumulator row each.
#pragma once
#include <cuda_fp16.h>
#include <cstdint>

#include "gm_device.cuh"

namespace gm {
namespace tc {

constexpr int kTileR = 4, kTileC = 32;      // output tile of one lane (8 x 16 also builds: measured slower, see above)
constexpr int kRowsPerLd = 32 / kTileC;     // accumulator rows in one 32-column tensor-memory load
constexpr int kSide = 128;                  // cutout side this engine is built for (128 lanes)
constexpr int kPitch = kSide;               // words per image row in shared memory (16-byte chunks XOR-swizzled, see swz)
constexpr int kNBuf = 3;                    // window-row buffers in tensor memory
constexpr int kMaxRing = 12;                // tap-row slots per ring at most; two rings (low / high tap rows)
constexpr int kMaxSlots = 2 * kMaxRing;
constexpr size_t kSmemLimit = 232448;       // 227 KB of dynamic shared memory per CTA

// Word offset of pixel (row R, column c), c a multiple of 4, in an image stored with `pitch` words per row
// (a multiple of 32): the 16-byte chunk index is XORed with three bits of row / kTileR, so that the eight lanes of
// a shared-memory wavefront, which read the same chunk of rows kTileR apart, hit eight different bank groups.
__host__ __device__ constexpr int swz_of(int R) { return (R / kTileR) & 7; }
__host__ __device__ constexpr int swz(int R, int c, int pitch) { return R * pitch + ((((c >> 2) ^ swz_of(R))) << 2); }
constexpr int kMmaWarps = 4;                // accumulator rows w, w + 4, ... each (one row at kTileR = 4)
constexpr int kAccPerWarp = kTileR / kMmaWarps;
constexpr int kThreads = (8 + kMmaWarps + 1) * 32;

template <int KP> struct Cfg {
  static_assert(((KP - 1) / 2) % 4 == 0, "half width must be a multiple of 4 (16-byte window chunks)");
  static constexpr int h = (KP - 1) / 2;
  static constexpr int NCH = (kTileC + KP - 1 + 15) / 16;     // 16-column chunks of a window row
  static constexpr int NY = kTileR + KP - 1;                  // window rows
  static constexpr int NR = 16 * (NCH - 1) + kTileC;          // rows of E_a
  static constexpr int kTapBytes = 2 * 2 * NR * 16;           // (hi, lo) x 2 k-blocks x NR rows x 8 halves
  static constexpr int kACols = NCH * 16;                     // tensor-memory columns of one row buffer
  static constexpr int kDCols = kTileR * kTileC;              // 128 accumulator columns per cutout
  static constexpr int kSlotWords = (kSide + 1) * kPitch;     // image rows + the zero row
  // tap-row ring depth: what two image slots leave of the shared memory, at least kTileR + 1 (kTileR tap rows are live per side)
  static constexpr int kRing = ((kSmemLimit - 2048 - 2 * (size_t)kSlotWords * 4) / (2 * (size_t)kTapBytes)) >= (size_t)kMaxRing
                                   ? kMaxRing : (int)((kSmemLimit - 2048 - 2 * (size_t)kSlotWords * 4) / (2 * (size_t)kTapBytes));
  static_assert(kRing >= kTileR + 1, "tap-row rings");
  static constexpr int kNSlot = 2 * kRing;
  // Window rows are visited OUTSIDE-IN (0, NY-1, 1, NY-2, ...): the tensor core adds every MMA into the
  // fp32 accumulator with truncation, a loss of half an ulp OF THE RUNNING SUM per step, so the tap rows
  // near the PSF centre, which carry most of the sum, must come last (measured: relative bias of a
  // convolved pixel -1.2e-5 in row order at K = 41).  A tap row serves window rows ta .. ta + kTileR - 1; it lives
  // in the LOW ring when its first use in that order is on the ascending side (window row ta at step 2 ta), in the
  // HIGH ring when it is on the descending side (window row ta + kTileR - 1 at step 2 (NY - ta - kTileR) + 1), i.e.
  // from ta = NY / 2 - kTileR / 2 + 1 on.  The tap-row producer issues every row at the step of its first use, and
  // with more than kTileR - 1 slots per ring the previous tenant of a slot has seen its last use by then: the MMA
  // warps never wait for a row whose slot they still hold (they did, with the rings split at NY / 2 and 8-row tiles).
  static constexpr int kSplit = NY / 2;
  static constexpr int kNLowRaw = kSplit - kTileR / 2 + 1;
  static constexpr int kNLow = kNLowRaw < 0 ? 0 : (kNLowRaw < KP ? kNLowRaw : KP);     // tap rows 0 .. kNLow-1
  static constexpr int kNHigh = KP - kNLow;                   // tap rows KP-1 down to kNLow
  __host__ __device__ static constexpr int seq(int i) { return (i & 1) ? NY - 1 - (i >> 1) : (i >> 1); }
  // ring slot of tap row ta and how many tap rows of one cutout were in that slot before it / in total
  // (RING = slots per ring of the kernel at hand)
  template <int RING> __host__ __device__ static constexpr int slot_of(int ta) { return ta < kNLow ? ta % RING : RING + (KP - 1 - ta) % RING; }
  template <int RING> __host__ __device__ static constexpr int index_in_slot(int ta) { return ta < kNLow ? ta / RING : (KP - 1 - ta) / RING; }
  template <int RING> __host__ __device__ static constexpr int uses_of_slot(int s) {
    return s < RING ? (kNLow - s + RING - 1) / RING : (kNHigh - (s - RING) + RING - 1) / RING;
  }
  static constexpr size_t kSmem = 2048 + 2 * (size_t)kSlotWords * 4 + (size_t)kNSlot * kTapBytes;
  static_assert(kSmem <= kSmemLimit, "shared memory");
  static_assert(2 * kDCols + kNBuf * kACols <= 512, "tensor memory");
};

struct ConvArgs {
  int B;                      // cutouts, each kSide x kSide
  const float* in;            // [B, 128, 128]
  float* out;                 // [B, 128, 128]
  const uint8_t* btab;        // [n_psf][KP tap rows][kTapBytes]: E_a of every tap row (k_tc_btab)
  const float* bscale;        // [n_psf]: 1 / (power-of-two scale of the PSF)
  long long btab_stride;      // bytes between the tables of consecutive cutouts (0: one PSF for all)
};

// ---- PTX wrappers ---------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(done) : "r"(bar), "r"(parity) : "memory");
  } while (!done);
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// one elected lane of the (converged) warp issues; every lane must execute these
__device__ __forceinline__ void mma_f16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t.reg .pred p, q;\n\t"
      "elect.sync _|q, 0xffffffff;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "@q tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
      ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(acc) : "memory");
}
// the same with the descriptor as (lo, hi) words: only lo (the start address field) changes between MMAs
__device__ __forceinline__ void mma_f16_ts2(uint32_t d_tmem, uint32_t a_tmem, uint32_t b_lo, uint32_t b_hi, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t.reg .pred p, q;\n\t.reg .b64 bd;\n\t"
      "mov.b64 bd, {%2, %3};\n\t"
      "elect.sync _|q, 0xffffffff;\n\t"
      "setp.ne.b32 p, %5, 0;\n\t"
      "@q tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], bd, %4, p;\n\t}"
      ::"r"(d_tmem), "r"(a_tmem), "r"(b_lo), "r"(b_hi), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void mma_commit(uint32_t bar) {
  asm volatile(
      "{\n\t.reg .pred q;\n\t"
      "elect.sync _|q, 0xffffffff;\n\t"
      "@q tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n\t}" ::"r"(bar) : "memory");
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
  return v;
}
__device__ __forceinline__ void sts128(uint32_t addr, uint4 v) {
  asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t (&v)[8]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr), "r"(v[0]), "r"(v[1]),
               "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
        "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
        "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
        "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr) : "memory");
}

// shared-memory matrix descriptor: K-major, no swizzle; element (row n, k) of the operand at
// start + (n % 8) * 16 + (n / 8) * SBO + (k % 8) * 2 + (k / 8) * LBO bytes
__host__ __device__ constexpr uint64_t smem_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16) |
         ((uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32) | ((uint64_t)1 << 46);
}
// instruction descriptor: fp16 x fp16 -> fp32, both operands K-major, M x N
__host__ __device__ constexpr uint32_t instr_desc(int M, int N) {
  return (1u << 4) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

// exact power-of-two scale that brings `amax` into [2^14, 2^15) (fp16 overflows at 65504)
__host__ __device__ inline float pow2_scale(float amax) {
  if (!(amax > 0.0f) || !(amax < 3.0e38f)) return 1.0f;
  int e;
#ifdef __CUDA_ARCH__
  e = ((__float_as_int(amax) >> 23) & 0xff) - 127;        // floor(log2) for normal numbers
  if (e < -100) e = -100;
  return __int_as_float((127 + 14 - e) << 23);
#else
  frexpf(amax, &e);                                        // amax = f * 2^e, f in [0.5, 1)
  e -= 1;
  if (e < -100) e = -100;
  return ldexpf(1.0f, 14 - e);
#endif
}
__device__ __forceinline__ uint32_t split_pack(float x) {  // (hi, lo) fp16 pair of x: lo half = hi part
  const __half hi = __float2half_rn(x);
  const __half lo = __float2half_rn(x - __half2float(hi));
  return (uint32_t)__half_as_ushort(hi) | ((uint32_t)__half_as_ushort(lo) << 16);
}

// ---- E_a tables -----------------------------------------------------------------------
// out[psf][a][part][kb][rho][e] (fp16) = part of s * Pf[a][8 kb + e - (rho - 16 (NCH - 1))], 0 outside the PSF;
// Pf = the PSF flipped in both axes (flip != 0: true convolution) or as given (adjoint).
template <int KP>
__global__ void __launch_bounds__(256) k_tc_btab(const float* __restrict__ psf, long long psf_stride, int K, int flip,
                                                 uint8_t* __restrict__ tab, float* __restrict__ bscale) {
  using C = Cfg<KP>;
  __shared__ float red[8];
  __shared__ float s_scale;
  const int ipsf = blockIdx.x / KP, a = blockIdx.x - ipsf * KP;   // one CTA per (PSF, tap row)
  const float* p = psf + (long long)ipsf * psf_stride;
  const int off = (KP - K) / 2;                            // a smaller PSF sits in the middle of the KP x KP frame
  float amax = 0.0f;
  for (int i = threadIdx.x; i < K * K; i += 256) amax = fmaxf(amax, fabsf(p[i]));
  for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = amax;
  __syncthreads();
  if (threadIdx.x == 0) {
    float m = 0.0f;
    for (int w = 0; w < 8; ++w) m = fmaxf(m, red[w]);
    s_scale = pow2_scale(m);
    if (a == 0) bscale[ipsf] = 1.0f / s_scale;
  }
  __syncthreads();
  const float s = s_scale;
  constexpr int per_a = C::kTapBytes / 2;                  // halves per tap row
  __half* out = reinterpret_cast<__half*>(tab + ((size_t)ipsf * KP + a) * C::kTapBytes);
  const int aa = (flip ? KP - 1 - a : a) - off;
  for (int idx = threadIdx.x; idx < per_a; idx += 256) {
    int r = idx;
    const int part = r / (2 * C::NR * 8); r -= part * (2 * C::NR * 8);
    const int kb = r / (C::NR * 8); r -= kb * (C::NR * 8);
    const int rho = r >> 3, e = r & 7;
    const int b = 8 * kb + e - (rho - 16 * (C::NCH - 1));
    float v = 0.0f;
    if (b >= 0 && b < KP) {
      const int bb = (flip ? KP - 1 - b : b) - off;
      if (aa >= 0 && aa < K && bb >= 0 && bb < K) v = p[aa * K + bb] * s;
    }
    const __half hi = __float2half_rn(v);
    out[idx] = part == 0 ? hi : __float2half_rn(v - __half2float(hi));
  }
}

// barrier indices of k_tc_conv (8 bytes each, from the start of the CTA's barrier area)
enum { IMG_FULL = 0, IMG_EMPTY = 2, A_FULL = 4, A_EMPTY = 4 + kNBuf, B_FULL = 4 + 2 * kNBuf, B_EMPTY = B_FULL + kMaxSlots,
       D_FULL = B_EMPTY + kMaxSlots, D_EMPTY = D_FULL + 2, N_BARS = D_EMPTY + 2 };
static_assert(N_BARS <= 64, "barrier area");

// MMA issue of accumulator rows R0, R0 + kMmaWarps, ... (NACC of them; one converged warp)
template <int KP, int R0, int NACC>
__device__ __forceinline__ void mma_role(int n_gal, uint32_t bars, uint32_t ring_addr, uint32_t tD, uint32_t tA) {
  using C = Cfg<KP>;
  constexpr uint32_t idesc = instr_desc(128, kTileC), idesc_half = instr_desc(128, kTileC / 2);
  constexpr uint32_t desc_hi = (uint32_t)(smem_desc(0, C::NR * 16, 128) >> 32);
  constexpr uint32_t desc_lo0 = (uint32_t)(smem_desc(0, C::NR * 16, 128) & 0xffffffffu);    // LBO field
  auto bar = [&](int i) -> uint32_t { return bars + 8u * (uint32_t)i; };
  int row_count = 0;
  for (int it = 0; it < n_gal; ++it) {
    const int d = it & 1;
    mbar_wait(bar(D_EMPTY + d), ((it >> 1) & 1) ^ 1);
    fence_after();
    uint32_t started = 0;                                         // bit rr: accumulator R0 + rr holds a sum already
#pragma unroll 1
    for (int i = 0; i < C::NY; ++i, ++row_count) {
      const int y = C::seq(i);
      const int buf = row_count % kNBuf;
      mbar_wait(bar(A_FULL + buf), (row_count / kNBuf) & 1);
      fence_after();
      const uint32_t acol = tA + (uint32_t)(buf * C::kACols);
#pragma unroll
      for (int rr = 0; rr < NACC; ++rr) {
        const int ta = y - (R0 + kMmaWarps * rr);                   // tap row
        if (ta < 0 || ta >= KP) continue;
        const int slot = C::template slot_of<C::kRing>(ta);
        mbar_wait(bar(B_FULL + slot), (uint32_t)(it * C::template uses_of_slot<C::kRing>(slot) + C::template index_in_slot<C::kRing>(ta)) & 1);
        fence_after();
        const uint32_t dcol = tD + (uint32_t)(d * C::kDCols + (R0 + kMmaWarps * rr) * kTileC);
        // start-address field of the hi part's chunk 0 (+ the constant LBO field); parts and chunks differ by constants
        const uint32_t lo0 = desc_lo0 + ((ring_addr + (uint32_t)(slot * C::kTapBytes)) >> 4);
        // chunk 0 reaches only the lower half of the output columns (j <= c) and the last chunk only the upper half
        // (j >= c - K + 1 >= kTileC / 2): those two run as N = kTileC / 2 MMAs; a full chunk goes first and overwrites
        static_assert(C::NCH >= 3 && 16 * (C::NCH - 1) - (KP - 1) >= kTileC / 2 && kTileC / 2 >= 16, "half-width edge chunks");
#pragma unroll
        for (int q = 0; q < C::NCH; ++q) {
          const int kc = q < C::NCH - 2 ? q + 1 : (q == C::NCH - 2 ? 0 : C::NCH - 1);       // 1 .. NCH-2, then 0, then NCH-1
          const bool lower = kc == 0, upper = kc == C::NCH - 1;
          const uint32_t b_hi = lo0 + (uint32_t)(16 * (C::NCH - 1 - kc) + (upper ? kTileC / 2 : 0));
          const uint32_t b_lo = b_hi + (uint32_t)(2 * C::NR);
          const uint32_t dc = dcol + (upper ? kTileC / 2 : 0);
          const uint32_t id = (lower || upper) ? idesc_half : idesc;
          mma_f16_ts2(dc, acol + kc * 16, b_hi, desc_hi, id, q ? 1u : ((started >> rr) & 1u));          // hi * hi (the first MMA overwrites)
          mma_f16_ts2(dc, acol + kc * 16 + 8, b_hi, desc_hi, id, 1);                   // lo * hi
          mma_f16_ts2(dc, acol + kc * 16, b_lo, desc_hi, id, 1);                       // hi * lo
        }
        started |= 1u << rr;
        mma_commit(bar(B_EMPTY + slot));
      }
      mma_commit(bar(A_EMPTY + buf));
    }
    mma_commit(bar(D_FULL + d));
  }
}

// ---- the convolution ------------------------------------------------------------------
template <int KP>
__global__ void __launch_bounds__(kThreads, 1) k_tc_conv(const ConvArgs a) {
  using C = Cfg<KP>;
  constexpr int h = C::h;
  extern __shared__ unsigned char smem_raw[];
  // carve: [barriers + scalars | 2 image slots | tap-row ring], the ring 1024-byte aligned
  unsigned char* base = reinterpret_cast<unsigned char*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint64_t* bars = reinterpret_cast<uint64_t*>(base);                 // 64 barriers at most
  uint32_t* tmem_base_s = reinterpret_cast<uint32_t*>(base + 512);
  float* inv_scale_s = reinterpret_cast<float*>(base + 528);          // [2]
  float* red_s = reinterpret_cast<float*>(base + 544);                // [4]
  unsigned char* ring = base + 1024;
  uint32_t* slots = reinterpret_cast<uint32_t*>(ring + (size_t)C::kNSlot * C::kTapBytes);

  static_assert(C::NY % 2 == 0, "outside-in order pairs the window rows");
  auto bar = [&](int i) -> uint32_t { return smem_u32(bars + i); };

  // warp index through a lane-0 broadcast: the compiler then knows it is warp-uniform and keeps the role
  // code (MMA descriptors, barrier addresses) in uniform registers
  const int tid = threadIdx.x, wid = __shfl_sync(0xffffffffu, tid >> 5, 0), lane = tid & 31;
  if (tid == 0) {
    for (int i = 0; i < 2; ++i) { mbar_init(bar(IMG_FULL + i), 4); mbar_init(bar(IMG_EMPTY + i), 4); }
    for (int i = 0; i < kNBuf; ++i) { mbar_init(bar(A_FULL + i), 4); mbar_init(bar(A_EMPTY + i), kMmaWarps); }
    for (int i = 0; i < C::kNSlot; ++i) { mbar_init(bar(B_FULL + i), 1); mbar_init(bar(B_EMPTY + i), kTileR); }
    for (int i = 0; i < 2; ++i) { mbar_init(bar(D_FULL + i), kMmaWarps); mbar_init(bar(D_EMPTY + i), 4); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (wid == 8 + kMmaWarps) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_base_s)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  // the zero rows of both slots (row kSide) and, once, everything else (skew gaps are read as padding)
  for (int i = tid; i < 2 * C::kSlotWords; i += kThreads) slots[i] = 0u;
  fence_before();
  __syncthreads();
  fence_after();
  const uint32_t tm = __shfl_sync(0xffffffffu, *tmem_base_s, 0);      // warp-uniform for the compiler
  const uint32_t tD = tm, tA = tm + 2 * C::kDCols;
  const int n_gal = (a.B - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;   // cutouts blockIdx.x, + gridDim.x, ...

  if (wid < 4) {
    // ------------------------- window rows -> tensor memory --------------------------
    // tensor-memory lane m = 32 w + t owns tile (row block m % kTRC, column block m / kTRC) of kTileR x kTileC pixels
    const uint32_t lane_base = (uint32_t)(32 * wid) << 16;
    constexpr int kTRC = kSide / kTileR;
    const int m = 32 * wid + lane, tr = m % kTRC, tc = m / kTRC;
    int row_count = 0;
    for (int it = 0; it < n_gal; ++it) {
      const int s = it & 1;
      const uint32_t slot = smem_u32(slots + (size_t)s * C::kSlotWords);       // byte address in shared memory
      const uint32_t zero = slot + 4u * (kSide * kPitch);
      mbar_wait(bar(IMG_FULL + s), (it >> 1) & 1);
      for (int i = 0; i < C::NY; ++i, ++row_count) {
        const int y = C::seq(i);
        const int buf = row_count % kNBuf;
        mbar_wait(bar(A_EMPTY + buf), ((row_count / kNBuf) & 1) ^ 1);
        fence_after();
        const int R = kTileR * tr + y - h;
        const bool row_ok = (unsigned)R < (unsigned)kSide;
        const uint32_t rowp = slot + 4u * (uint32_t)(R * kPitch);
        const int sw = swz_of(R);
#pragma unroll
        for (int kc = 0; kc < C::NCH; ++kc) {
          uint32_t w[16];
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const int c0 = kTileC * tc - h + 16 * kc + 4 * q;
            const uint4 v = lds128((row_ok && (unsigned)c0 < (unsigned)kSide) ? rowp + 16u * (uint32_t)((c0 >> 2) ^ sw) : zero);
            w[4 * q] = v.x; w[4 * q + 1] = v.y; w[4 * q + 2] = v.z; w[4 * q + 3] = v.w;
          }
          uint32_t hi[8], lo[8];
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            hi[j] = __byte_perm(w[2 * j], w[2 * j + 1], 0x5410);
            lo[j] = __byte_perm(w[2 * j], w[2 * j + 1], 0x7632);
          }
          const uint32_t col = tA + (uint32_t)(buf * C::kACols + kc * 16) + lane_base;
          tmem_st8(col, hi);
          tmem_st8(col + 8, lo);
        }
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(A_FULL + buf));
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(IMG_EMPTY + s));
    }
  } else if (wid < 8) {
    // ------------------- cutout loader and accumulator drain -------------------------
    const int lw = wid - 4, ltid = tid - 128;
    const uint32_t lane_base = (uint32_t)(32 * lw) << 16;
    auto drain = [&](int it) {
      const int d = it & 1;
      const int g = (int)blockIdx.x + it * (int)gridDim.x;
      mbar_wait(bar(D_FULL + d), (it >> 1) & 1);
      fence_after();
      const float inv = inv_scale_s[d] * a.bscale[a.btab_stride ? g : 0];
      float* outp = a.out + (size_t)g * kSide * kSide;
      constexpr int kTRC = kSide / kTileR;
      const int m = 32 * lw + lane, tr = m % kTRC, tc = m / kTRC;
#pragma unroll 1
      for (int q = 0; q < C::kDCols / 32; ++q) {                     // 32 columns = kRowsPerLd accumulator rows
        uint32_t v[32];
        tmem_ld32(tD + (uint32_t)(d * C::kDCols + 32 * q) + lane_base, v);
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const int r = kRowsPerLd * q + (4 * k) / kTileC, c = (4 * k) % kTileC;
          *reinterpret_cast<float4*>(outp + (size_t)(kTileR * tr + r) * kSide + kTileC * tc + c) =
              make_float4(__uint_as_float(v[4 * k]) * inv, __uint_as_float(v[4 * k + 1]) * inv,
                          __uint_as_float(v[4 * k + 2]) * inv, __uint_as_float(v[4 * k + 3]) * inv);
        }
      }
      fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(D_EMPTY + d));
    };
    for (int it = 0; it < n_gal; ++it) {
      const int s = it & 1;
      const int g = (int)blockIdx.x + it * (int)gridDim.x;
      const uint32_t slot = smem_u32(slots + (size_t)s * C::kSlotWords);
      mbar_wait(bar(IMG_EMPTY + s), ((it >> 1) & 1) ^ 1);
      // pass 1: global fp32 -> the slot (as fp32), and the largest magnitude of the cutout
      const float4* src = reinterpret_cast<const float4*>(a.in + (size_t)g * kSide * kSide);
      float amax = 0.0f;
#pragma unroll 4
      for (int i = ltid; i < kSide * kSide / 4; i += 128) {
        const float4 v = __ldg(src + i);
        const int R = i >> 5, c = (i & 31) << 2;
        sts128(slot + 4u * (uint32_t)swz(R, c, kPitch),
               make_uint4(__float_as_uint(v.x), __float_as_uint(v.y), __float_as_uint(v.z), __float_as_uint(v.w)));
        amax = fmaxf(fmaxf(amax, fmaxf(fabsf(v.x), fabsf(v.y))), fmaxf(fabsf(v.z), fabsf(v.w)));
      }
      for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
      if (lane == 0) red_s[lw] = amax;
      asm volatile("bar.sync 1, 128;" ::: "memory");
      const float sc = pow2_scale(fmaxf(fmaxf(red_s[0], red_s[1]), fmaxf(red_s[2], red_s[3])));
      // pass 2: every thread turns its own pixels into (hi, lo) fp16 pairs in place
#pragma unroll 4
      for (int i = ltid; i < kSide * kSide / 4; i += 128) {
        const int R = i >> 5, c = (i & 31) << 2;
        const uint32_t p = slot + 4u * (uint32_t)swz(R, c, kPitch);
        const uint4 v = lds128(p);
        sts128(p, make_uint4(split_pack(__uint_as_float(v.x) * sc), split_pack(__uint_as_float(v.y) * sc),
                             split_pack(__uint_as_float(v.z) * sc), split_pack(__uint_as_float(v.w) * sc)));
      }
      asm volatile("bar.sync 1, 128;" ::: "memory");              // red_s may be rewritten after this
      if (ltid == 0) inv_scale_s[s] = 1.0f / sc;                     // read by drain(it), after the next bar.sync
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(IMG_FULL + s));                 // the window rows of cutout `it` may start
      if (it > 0) drain(it - 1);                                     // reads inv_scale_s[(it - 1) & 1]
    }
    if (n_gal > 0) {
      asm volatile("bar.sync 1, 128;" ::: "memory");              // inv_scale_s of the last cutout is visible
      drain(n_gal - 1);
    }
  } else if (wid < 8 + kMmaWarps) {
    // ----------------------------------- MMA issue ------------------------------------
    // (the accumulator pair is a template argument so that every address of the issue loop is
    // warp-uniform at compile time and stays in uniform registers)
    static_assert(kMmaWarps == 4, "accumulator rows w, w + 4 per MMA warp");
    if (wid == 8) mma_role<KP, 0, kAccPerWarp>(n_gal, smem_u32(bars), smem_u32(ring), tD, tA);
    else if (wid == 9) mma_role<KP, 1, kAccPerWarp>(n_gal, smem_u32(bars), smem_u32(ring), tD, tA);
    else if (wid == 10) mma_role<KP, 2, kAccPerWarp>(n_gal, smem_u32(bars), smem_u32(ring), tD, tA);
    else mma_role<KP, 3, kAccPerWarp>(n_gal, smem_u32(bars), smem_u32(ring), tD, tA);
  } else {
    // ------------------------------- tap-row producer --------------------------------
    // in the order of first use: window row y = seq(i) brings tap row y (r = 0) on the low side and
    // tap row y - 3 (r = 3) on the high side
    if (lane == 0) {
      for (int it = 0; it < n_gal; ++it) {
        const int g = (int)blockIdx.x + it * (int)gridDim.x;
        const uint8_t* tab = a.btab + (size_t)g * a.btab_stride;
        for (int i = 0; i < C::NY; ++i) {
          const int y = C::seq(i);
          const int ta = (i & 1) ? y - (kTileR - 1) : y;
          if ((i & 1) ? (ta < C::kNLow || ta >= KP) : (ta >= C::kNLow)) continue;
          const int slot = C::template slot_of<C::kRing>(ta);
          const uint32_t gen = (uint32_t)(it * C::template uses_of_slot<C::kRing>(slot) + C::template index_in_slot<C::kRing>(ta));
          mbar_wait(bar(B_EMPTY + slot), (gen & 1) ^ 1);
          mbar_expect_tx(bar(B_FULL + slot), C::kTapBytes);
          bulk_g2s(smem_u32(ring + (size_t)slot * C::kTapBytes), tab + (size_t)ta * C::kTapBytes, C::kTapBytes, bar(B_FULL + slot));
        }
      }
    }
  }
  fence_before();
  __syncthreads();
  if (wid == 8 + kMmaWarps) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tm) : "memory");
}

}  // namespace tc
}  // namespace gm
