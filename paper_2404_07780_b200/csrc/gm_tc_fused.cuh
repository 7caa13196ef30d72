// gm_tc_fused.cuh -- steps a1..a5 of the hot path for 64 / 96 / 128 px cutouts with BOTH convolutions on the
// tensor cores (the engine of gm_tc.cuh): one persistent CTA per SM, two cutouts in flight, nothing but
// chi^2 and the kNSum partial sums per component leaving the SM (mode 0 writes the model image).
//
// Roles (4 + HW + 4 + 1 warps, all hand-offs by mbarrier / named barrier):
//   warps 0-3        window rows of the current job: shared memory -> tensor memory (A operand)
//   HW helper warps  a1 render S into a slot, scale + split into (hi, lo) fp16 pairs; after the forward
//                    convolution drain M (tensor memory -> slot, fp32), a3 residual / chi^2 / G in place, scale +
//                    split G; after the adjoint convolution drain A, a5 gradient sums
//   4 MMA warps      MMA issue, one accumulator row of the 4 x 32 tiles each
//   last warp        streams the Toeplitz band blocks E_a (forward or adjoint table) through the two rings
// A JOB is one convolution of one cutout.  Jobs run in the order C1(a) C1(b) C2(a) C2(b) (cutouts a, b in
// slots 0, 1), so the helpers always work on the slot the tensor cores are not reading: the same
// schedule as k_fused (gm_fused.cuh), with the FFMA2 loop replaced by tcgen05.mma.
#pragma once
#include "gm_kernels.cuh"
#include "gm_tc.cuh"

namespace gm {
namespace tc {

// Helper warps: k_tc_fused overlaps them with the tensor pipe of the other slot, and more than 8 only add traffic
// on the shared-memory pipe that binds it (measured: 16 warps K = 41 +18 %, K = 25 +1 %); the one-slot super-tile
// kernels run their fill phase alone, where 16 warps are 1.5x faster (C4 -13 %, C2 -8 %).
template <int HW> struct Roles {
  static_assert(HW == 8 || HW == 16, "helper warps: a multiple of 4 (tensor-memory lane quarters)");
  static constexpr int kHelp = HW;
  static constexpr int kThreads = (4 + HW + kMmaWarps + 1) * 32;
  static constexpr int kHN = 32 * HW;
  static constexpr int kLdPerWarp = 4 / (HW / 4);             // 32-column accumulator loads (of 4 per lane) one helper warp drains
  static constexpr int kLastWarp = 4 + HW + kMmaWarps;
  // header of the shared memory: 64 barriers, the tensor-memory base, reduction scratch [HW * kNSum] + [HW] maxima
  static constexpr int kHeaderBytes = (528 + (HW * kNSum + HW) * 4 + 127) / 128 * 128;
};
constexpr int kAlignSlack = 128;                              // the dynamic shared memory is re-aligned to 128 bytes
constexpr int kFusedHW = 8, kTileHW = 16;

struct FusedTcArgs {
  ModelDesc md;
  int B;
  int mode;                  // 0 render (write M), 1 chi^2 only, 2 chi^2 + gradient
  const CompConst* cc;
  const uint8_t* btab_fwd; const uint8_t* btab_adj;   // E_a tables of the flipped PSF and of the PSF as given
  long long btab_stride;     // bytes between the tables of consecutive galaxies (0: one PSF for the batch)
  const float* bscale;       // [n_psf] 1 / (power-of-two scale of the PSF)
  const float* data; const float* sigma; const uint8_t* mask;
  float* out;                // mode 0: model image [B,128,128]
  int any_unconv;            // the model has components that do not go through the PSF (R:C3; the sky is one)
  float* gseed;              // [B,SIDE,SIDE] back-seed G for the gradient of those components (mode 2 with any_unconv)
  float* chi2_part;          // [B]
  float* grad_part;          // [B, n_comp, kNSum]
  const int* frozen;
  const int* live; const int* n_live;
  unsigned long long* trace; // gm_trace_set: phase time stamps of CTA 0 (measurement hook), or nullptr
};

// ---- phase trace (gm_trace_set, include/gm.h): CTA 0 appends (tag << 48 | clock64) records, one list per role ----
constexpr int kTraceCap = 2048;                 // records per role
enum { TR_HELPER = 0, TR_MMA = 1, TR_WINDOW = 2, TR_ROLES = 3 };
enum { TR_PRODUCE = 1, TR_PRODUCE_END, TR_DRAIN_WAIT, TR_DRAIN, TR_RESIDUAL, TR_RESIDUAL_END, TR_GRADIENT, TR_GRADIENT_END,
       TR_JOB, TR_JOB_END };
struct Tracer {
  unsigned long long* p = nullptr;
  int n = 0;
  __device__ __forceinline__ void init(unsigned long long* base, int role, bool me) {
    p = (base && blockIdx.x == 0 && me) ? base + (size_t)role * kTraceCap : nullptr;
  }
  __device__ __forceinline__ void ev(int tag, int item) {
    if (p && n < kTraceCap) {
      unsigned long long t;
      asm volatile("mov.u64 %0, %%clock64;" : "=l"(t));
      p[n++] = ((unsigned long long)((tag << 8) | (item & 255)) << 48) | (t & 0xffffffffffffull);
    }
  }
};

enum { F_IN_FULL = 0, F_D_FULL = 2, F_A_FULL = 4, F_A_EMPTY = 4 + kNBuf, F_B_FULL = 4 + 2 * kNBuf, F_B_EMPTY = F_B_FULL + kMaxSlots,
       F_SLOT_FREE = F_B_EMPTY + kMaxSlots, F_N_BARS = F_SLOT_FREE + 1 };
static_assert(F_N_BARS <= 64, "barrier area");

// the jobs of one CTA in tensor-core order; f(item, phase, slot)
template <typename F>
__device__ __forceinline__ void for_each_job(int n_items, int phases, F&& f) {
  for (int m = 0; 2 * m < n_items; ++m)
    for (int ph = 0; ph < phases; ++ph)
      for (int s = 0; s < 2; ++s) {
        const int item = 2 * m + s;
        if (item < n_items) f(item, ph, s);
      }
}

// MMA issue of accumulator rows R0 and R0 + kMmaWarps for every job (one converged warp); RING = tap-row slots per ring
template <int KP, int R0, int RING>
__device__ __forceinline__ void fused_mma_role(int n_items, int phases, uint32_t bars, uint32_t ring_addr, uint32_t tD, uint32_t tA,
                                               unsigned long long* trace = nullptr) {
  using C = Cfg<KP>;
  constexpr uint32_t idesc = instr_desc(128, kTileC), idesc_half = instr_desc(128, kTileC / 2);
  constexpr uint32_t desc_hi = (uint32_t)(smem_desc(0, C::NR * 16, 128) >> 32);
  constexpr uint32_t desc_lo0 = (uint32_t)(smem_desc(0, C::NR * 16, 128) & 0xffffffffu);
  auto bar = [&](int i) -> uint32_t { return bars + 8u * (uint32_t)i; };
  int row_count = 0, jc = 0;
  Tracer tr;
  tr.init(trace, TR_MMA, R0 == 0 && (threadIdx.x & 31) == 0);
  for_each_job(n_items, phases, [&](int item, int ph, int s) {
    uint32_t started = 0;                                  // bit rr: accumulator row R0 + kMmaWarps rr holds a sum already
    bool first_row = true;
#pragma unroll 1
    for (int i = 0; i < C::NY; ++i, ++row_count) {
      const int y = C::seq(i);
      const int buf = row_count % kNBuf;
      mbar_wait(bar(F_A_FULL + buf), (row_count / kNBuf) & 1);
      fence_after();
      if (first_row) { tr.ev(TR_JOB, 2 * item + ph); first_row = false; }      // the first window row of the job is there
      const uint32_t acol = tA + (uint32_t)(buf * C::kACols);
#pragma unroll
      for (int rr = 0; rr < kAccPerWarp; ++rr) {
        const int ta = y - (R0 + kMmaWarps * rr);
        if (ta < 0 || ta >= KP) continue;
        const int slot = C::template slot_of<RING>(ta);
        mbar_wait(bar(F_B_FULL + slot), (uint32_t)(jc * C::template uses_of_slot<RING>(slot) + C::template index_in_slot<RING>(ta)) & 1);
        fence_after();
        const uint32_t dcol = tD + (uint32_t)(s * C::kDCols + (R0 + kMmaWarps * rr) * kTileC);
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
        mma_commit(bar(F_B_EMPTY + slot));
      }
      mma_commit(bar(F_A_EMPTY + buf));
    }
    mma_commit(bar(F_D_FULL + s));
    tr.ev(TR_JOB_END, 2 * item + ph);                      // the last MMA of the job is issued (not yet complete)
    ++jc;
  });
}

// one window row of a lane's tile: NCH chunks of 16 columns, shared memory (hi, lo) words -> tensor memory.
// chunk0 = 16-byte chunk index of the window's first column in the row at `rowp` (may be negative / beyond n_chunks:
// those chunks and rows with !row_ok read the zero row); sw = swizzle of the row.
template <int KP>
__device__ __forceinline__ void stage_window_row(uint32_t rowp, uint32_t zero, bool row_ok, int chunk0, int n_chunks, int sw,
                                                 uint32_t tcol) {
  using C = Cfg<KP>;
#pragma unroll
  for (int kc = 0; kc < C::NCH; ++kc) {
    uint32_t w[16];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      // window columns beyond kTileC + KP - 2 meet only zero taps (chunk padding): zeros, no shared-memory read
      // (the shared-memory pipe is what this engine runs out of first, and these warps are its largest client)
      if (16 * kc + 4 * q >= kTileC + KP - 1) { w[4 * q] = w[4 * q + 1] = w[4 * q + 2] = w[4 * q + 3] = 0u; continue; }
      const int ch = chunk0 + 4 * kc + q;
      const uint4 v = lds128((row_ok && (unsigned)ch < (unsigned)n_chunks) ? rowp + 16u * (uint32_t)(ch ^ sw) : zero);
      w[4 * q] = v.x; w[4 * q + 1] = v.y; w[4 * q + 2] = v.z; w[4 * q + 3] = v.w;
    }
    uint32_t hi[8], lo[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      hi[j] = __byte_perm(w[2 * j], w[2 * j + 1], 0x5410);
      lo[j] = __byte_perm(w[2 * j], w[2 * j + 1], 0x7632);
    }
    tmem_st8(tcol + kc * 16, hi);
    tmem_st8(tcol + kc * 16 + 8, lo);
  }
}

// Geometry of k_tc_fused for square cutouts of SIDE = 64, 96 or 128 pixels: a cutout is (SIDE / kTileR) x (SIDE / kTileC)
// tiles; G = 4, 1, 1 cutouts share the 128 lanes of a pass (64 px: one lane quarter each; 96 px: 72 lanes used).
template <int KP, int SIDE> struct FusedGeomTc {
  using C = Cfg<KP>;
  static_assert(SIDE == 64 || SIDE == 96 || SIDE == 128, "cutout side");
  static constexpr int TRC = SIDE / kTileR, TCC = SIDE / kTileC, TPG = TRC * TCC;   // tile rows / columns / tiles per cutout
  static constexpr int G = 128 / TPG;                         // cutouts per pass
  static constexpr int W4 = SIDE / 4, kGroups = SIDE * W4;    // groups of four pixels per row / per cutout
  static constexpr int kCutWords = (SIDE + 1) * SIDE;         // rows + the zero row, pitch = SIDE words (XOR-swizzled chunks)
  static constexpr int kSlotWordsF = G * kCutWords;
  static constexpr size_t kFixed = kAlignSlack + Roles<kFusedHW>::kHeaderBytes + 2 * (size_t)kSlotWordsF * 4;     // alignment slack, header, slots
  static constexpr int kRingF = ((kSmemLimit - kFixed) / (2 * (size_t)C::kTapBytes)) >= (size_t)kMaxRing
                                    ? kMaxRing : (int)((kSmemLimit - kFixed) / (2 * (size_t)C::kTapBytes));
  static_assert(kRingF >= kTileR + 1, "tap-row rings");
  static constexpr size_t kSmem = kFixed + (size_t)(2 * kRingF) * C::kTapBytes;
  static_assert(kSmem <= kSmemLimit, "shared memory");
};

// UNCONV: the model has components that do not go through the PSF (a variant of its own: the extra tests in the
// helper loops cost 12 % at K = 25, where the helper warps bind)
template <int KP, int SIDE, bool UNCONV>
__global__ void __launch_bounds__(Roles<kFusedHW>::kThreads, 1) k_tc_fused(const FusedTcArgs a) {
  using C = Cfg<KP>;
  using Gm = FusedGeomTc<KP, SIDE>;
  using Ro = Roles<kFusedHW>;
  constexpr int h = C::h, G = Gm::G, kHN = Ro::kHN, kHelp = Ro::kHelp;
  extern __shared__ unsigned char smem_raw[];
  unsigned char* base = reinterpret_cast<unsigned char*>(((uintptr_t)smem_raw + (kAlignSlack - 1)) & ~(uintptr_t)(kAlignSlack - 1));
  uint64_t* bars = reinterpret_cast<uint64_t*>(base);
  uint32_t* tmem_base_s = reinterpret_cast<uint32_t*>(base + 512);
  float* red = reinterpret_cast<float*>(base + 528);                // [kHelp * kNSum] sums, then [kHelp] maxima
  float* redmax = red + kHelp * kNSum;
  unsigned char* ring = base + Ro::kHeaderBytes;
  uint32_t* slots = reinterpret_cast<uint32_t*>(ring + (size_t)(2 * Gm::kRingF) * C::kTapBytes);
  auto bar = [&](int i) -> uint32_t { return smem_u32(bars + i); };

  // a CTA without work (late iterations of a fit with early stop: a few live galaxies, 148 CTAs) leaves at once, before
  // it allocates tensor memory or zeroes 130 KB of slots: it would hold the SM against the other buckets' kernels
  if ((int)blockIdx.x >= (a.live ? *a.n_live : a.B)) return;
  // warp index through a lane-0 broadcast: warp-uniform for the compiler (uniform registers in the role code)
  const int tid = threadIdx.x, wid = __shfl_sync(0xffffffffu, tid >> 5, 0), lane = tid & 31;
  if (tid == 0) {
    for (int i = 0; i < 2; ++i) { mbar_init(bar(F_IN_FULL + i), kHelp); mbar_init(bar(F_D_FULL + i), kMmaWarps); }
    for (int i = 0; i < kNBuf; ++i) { mbar_init(bar(F_A_FULL + i), 4); mbar_init(bar(F_A_EMPTY + i), kMmaWarps); }
    for (int i = 0; i < 2 * Gm::kRingF; ++i) { mbar_init(bar(F_B_FULL + i), 1); mbar_init(bar(F_B_EMPTY + i), kTileR); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  constexpr int kLastWarp = Ro::kLastWarp;
  if (wid == kLastWarp) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_base_s)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  for (int i = tid; i < 2 * Gm::kSlotWordsF; i += Ro::kThreads) slots[i] = 0u;    // the zero rows
  fence_before();
  __syncthreads();
  fence_after();
  const uint32_t tm = __shfl_sync(0xffffffffu, *tmem_base_s, 0);
  const uint32_t tD = tm, tA = tm + 2 * C::kDCols;

  const bool with_grad = a.mode == 2;
  const int phases = with_grad ? 2 : 1;
  const int n_gal = a.live ? *a.n_live : a.B;
  // the galaxies of this CTA: entries blockIdx.x, + gridDim.x, ... of the list, G at a time (one item = one pass)
  const int n_k = (n_gal - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
  const int n_items = (n_k + G - 1) / G;
  auto galaxy = [&](int item, int g) -> int {              // -1: no galaxy in this place, or one that no longer iterates
    const int k = item * G + g;
    if (k >= n_k) return -1;
    const int i = (int)blockIdx.x + k * (int)gridDim.x;
    const int b = a.live ? a.live[i] : i;
    return (a.frozen && a.frozen[b]) ? -1 : b;
  };

  if (wid < 4) {
    // ------------------------- window rows -> tensor memory --------------------------
    const uint32_t lane_base = (uint32_t)(32 * wid) << 16;
    const int m = 32 * wid + lane;                         // lane of the tensor memory = tile (g, tr, tc)
    const int g = m / Gm::TPG, rem = m - g * Gm::TPG;
    const int tr = rem % Gm::TRC, tc = rem / Gm::TRC;
    const bool lane_ok = g < G;
    int row_count = 0, cnt[2] = {0, 0};
    for_each_job(n_items, phases, [&](int, int, int s) {
      const uint32_t cut = smem_u32(slots + (size_t)s * Gm::kSlotWordsF + (size_t)(lane_ok ? g : 0) * Gm::kCutWords);
      const uint32_t zero = cut + 4u * (SIDE * SIDE);
      mbar_wait(bar(F_IN_FULL + s), cnt[s] & 1);
      ++cnt[s];
      for (int i = 0; i < C::NY; ++i, ++row_count) {
        const int y = C::seq(i);
        const int buf = row_count % kNBuf;
        mbar_wait(bar(F_A_EMPTY + buf), ((row_count / kNBuf) & 1) ^ 1);
        fence_after();
        const int R = kTileR * tr + y - h;
        const bool row_ok = lane_ok && (unsigned)R < (unsigned)SIDE;
        stage_window_row<KP>(cut + 4u * (uint32_t)(R * SIDE), zero, row_ok, (kTileC * tc - h) >> 2, SIDE / 4, swz_of(R),
                             tA + (uint32_t)(buf * C::kACols) + lane_base);
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(F_A_FULL + buf));
      }
    });
  } else if (wid < 4 + kHelp) {
    // ------------------------------------ helpers -------------------------------------
    const int hw = wid - 4, htid = tid - 128;
    const uint32_t lane_base = (uint32_t)(32 * (hw & 3)) << 16;
    float inv_sc[2][G];                                    // 1 / scale of cutout g of slot s (every thread holds the same)
#pragma unroll
    for (int g = 0; g < G; ++g) inv_sc[0][g] = inv_sc[1][g] = 1.0f;
    int cnt_d[2] = {0, 0};
    Tracer tr;
    tr.init(a.trace, TR_HELPER, htid == 0);
    auto cut_addr = [&](int s, int g) -> uint32_t { return smem_u32(slots + (size_t)s * Gm::kSlotWordsF + (size_t)g * Gm::kCutWords); };
    auto px_addr = [&](uint32_t cut, int R, int c) -> uint32_t { return cut + 4u * (uint32_t)swz(R, c, SIDE); };
    auto help_sync = [&]() { asm volatile("bar.sync 1, %0;" ::"n"(kHN) : "memory"); };
    constexpr int W4 = Gm::W4, kGroups = Gm::kGroups;      // a warp walks whole rows: coalesced global, conflict-free shared

    // fp32 values of one cutout -> (hi, lo) fp16 pairs of value * 2^e, e from the largest magnitude `amax`
    // (every thread passes its own maximum; converts the groups it owns)
    auto scale_and_split = [&](uint32_t cut, float amax) -> float {
      for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
      if (lane == 0) redmax[hw] = amax;
      help_sync();
      float mx = redmax[0];
#pragma unroll
      for (int w = 1; w < kHelp; ++w) mx = fmaxf(mx, redmax[w]);
      const float sc = pow2_scale(mx);
#pragma unroll 2
      for (int idx = htid; idx < kGroups; idx += kHN) {
        const uint32_t p = px_addr(cut, idx / W4, (idx % W4) << 2);
        const uint4 v = lds128(p);
        sts128(p, make_uint4(split_pack(__uint_as_float(v.x) * sc), split_pack(__uint_as_float(v.y) * sc),
                             split_pack(__uint_as_float(v.z) * sc), split_pack(__uint_as_float(v.w) * sc)));
      }
      help_sync();                                         // redmax may be rewritten
      return 1.0f / sc;
    };
    auto signal_input = [&](int s) {
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(F_IN_FULL + s));
    };

    // a1: S of every cutout of the item (all components go through the PSF on this path) -> slot s
    auto produce = [&](int item, int s) {
      tr.ev(TR_PRODUCE, item);
#pragma unroll
      for (int g = 0; g < G; ++g) {
        const int b = galaxy(item, g);
        const uint32_t cut = cut_addr(s, g);
        float amax = 0.0f;
        if (b >= 0) {
          const CompConst* ccb = a.cc + (size_t)b * a.md.n_comp;
          int c_first = -1, c_last = -1;                   // the components that go through the PSF
          for (int c = 0; c < a.md.n_comp; ++c)
            if (!UNCONV || a.md.conv[c]) { if (c_first < 0) c_first = c; c_last = c; }
          if (c_first < 0)                                 // none: S = 0, the model is the unconvolved part alone
            for (int idx = htid; idx < kGroups; idx += kHN) sts128(px_addr(cut, idx / W4, (idx % W4) << 2), make_uint4(0u, 0u, 0u, 0u));
          for (int c = 0; c < a.md.n_comp; ++c) {
            if (UNCONV && !a.md.conv[c]) continue;
            const CompConst cc = ccb[c];
            const bool box = a.md.box[c] != 0;
            const bool first = c == c_first, last = c == c_last;
            dispatch_kind(a.md.kind[c], [&]<int KIND>() {
              for (int idx = htid; idx < kGroups; idx += kHN) {
                const int R = idx / W4, x = (idx % W4) << 2;
                float v[4];
                value4<KIND, kFastForward>(cc, box, (float)x + 0.5f, (float)SIDE - 0.5f - (float)R, v);   // R:G1
                const uint32_t p = px_addr(cut, R, x);
                if (!first) {
                  const uint4 q = lds128(p);
                  v[0] += __uint_as_float(q.x); v[1] += __uint_as_float(q.y); v[2] += __uint_as_float(q.z); v[3] += __uint_as_float(q.w);
                }
                if (last) amax = fmaxf(fmaxf(amax, fmaxf(fabsf(v[0]), fabsf(v[1]))), fmaxf(fabsf(v[2]), fabsf(v[3])));
                sts128(p, make_uint4(__float_as_uint(v[0]), __float_as_uint(v[1]), __float_as_uint(v[2]), __float_as_uint(v[3])));
              }
            });
          }
        } else {
          for (int idx = htid; idx < kGroups; idx += kHN) sts128(px_addr(cut, idx / W4, (idx % W4) << 2), make_uint4(0u, 0u, 0u, 0u));
        }
        if (!isfinite(amax)) amax = 0.0f;
        inv_sc[s][g] = scale_and_split(cut, amax);
      }
      signal_input(s);
      tr.ev(TR_PRODUCE_END, item);
    };

    // accumulators of the job on slot s -> the cutouts of the slot, as fp32
    auto drain = [&](int item, int s) {
      tr.ev(TR_DRAIN_WAIT, item);
      mbar_wait(bar(F_D_FULL + s), cnt_d[s] & 1);
      ++cnt_d[s];
      fence_after();
      tr.ev(TR_DRAIN, item);
      const int m = 32 * (hw & 3) + lane;                  // this thread's lane of the tensor memory
      const int g = m / Gm::TPG, rem = m - g * Gm::TPG;
      const int tr_ = rem % Gm::TRC, tc = rem / Gm::TRC;
      const bool lane_ok = g < G;
      const int b = lane_ok ? galaxy(item, g) : -1;
      float isc = 1.0f;
#pragma unroll
      for (int gg = 0; gg < G; ++gg) isc = (gg == g) ? inv_sc[s][gg] : isc;
      const float inv = isc * a.bscale[(a.btab_stride && b >= 0) ? b : 0];
      const uint32_t cut = cut_addr(s, lane_ok ? g : 0);
      const int q_first = Ro::kLdPerWarp * (hw >> 2);
#pragma unroll 1
      for (int q = q_first; q < q_first + Ro::kLdPerWarp; ++q) {    // 32 columns = kRowsPerLd accumulator rows
        uint32_t v[32];
        tmem_ld32(tD + (uint32_t)(s * C::kDCols + 32 * q) + lane_base, v);
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        if (lane_ok) {
#pragma unroll
          for (int k = 0; k < 8; ++k)
            sts128(px_addr(cut, kTileR * tr_ + kRowsPerLd * q + (4 * k) / kTileC, kTileC * tc + (4 * k) % kTileC),
                   make_uint4(__float_as_uint(__uint_as_float(v[4 * k]) * inv), __float_as_uint(__uint_as_float(v[4 * k + 1]) * inv),
                              __float_as_uint(__uint_as_float(v[4 * k + 2]) * inv), __float_as_uint(__uint_as_float(v[4 * k + 3]) * inv)));
        }
      }
      fence_before();
      help_sync();                                         // every image is in the slot
    };

    // a3: M (slot, fp32) -> chi^2 and G in place, then G as fp16 pairs for the adjoint convolution; mode 0 writes M out
    auto residual = [&](int item, int s) {
#pragma unroll
      for (int g = 0; g < G; ++g) {
        const int b = galaxy(item, g);
        const uint32_t cut = cut_addr(s, g);
        float chi2 = 0.0f, amax = 0.0f;
        if (b >= 0) {
          const size_t img = (size_t)b * SIDE * SIDE;
          // components that do not go through the PSF are added to the convolved image here (R:C3), pixel by pixel
          const CompConst* ccb = a.cc + (size_t)b * a.md.n_comp;
          auto add_unconv = [&](uint4& m4, int idx) {
            const int R = idx / W4, x = (idx % W4) << 2;
            const float y = (float)SIDE - 0.5f - (float)R;
            float m[4] = {__uint_as_float(m4.x), __uint_as_float(m4.y), __uint_as_float(m4.z), __uint_as_float(m4.w)};
            for (int c = 0; c < a.md.n_comp; ++c) {
              if (a.md.conv[c]) continue;
              const CompConst cc = ccb[c];
              const int kind = a.md.kind[c];
#pragma unroll
              for (int k = 0; k < 4; ++k) {
                const float U = (kind == GM_SKY) ? 1.0f : profile_value(kind, cc, geometry<false>(cc, a.md.box[c] != 0, (float)(x + k) + 0.5f, y).r);
                m[k] = fmaf(cc.amp, U, m[k]);
              }
            }
            m4 = make_uint4(__float_as_uint(m[0]), __float_as_uint(m[1]), __float_as_uint(m[2]), __float_as_uint(m[3]));
          };
          if (a.mode == 0) {
            for (int idx = htid; idx < kGroups; idx += kHN) {
              uint4 v = lds128(px_addr(cut, idx / W4, (idx % W4) << 2));
              if (UNCONV) add_unconv(v, idx);
              *reinterpret_cast<float4*>(a.out + img + 4 * (size_t)idx) =
                  make_float4(__uint_as_float(v.x), __uint_as_float(v.y), __uint_as_float(v.z), __uint_as_float(v.w));
            }
          } else {
            // branch free; the weight and the residual are SELECTED for unused pixels, never multiplied by 0 (R:X1)
            auto one = [&](float mm, float d, float sg, bool used) -> float {
              float w = rcp_fast(sg * sg), rho = d - mm;
              w = used ? w : 0.0f;
              rho = used ? rho : 0.0f;
              const float t = w * rho;
              chi2 = fmaf(t, rho, chi2);
              const float gg = -2.0f * t;
              amax = fmaxf(amax, fabsf(gg));
              return gg;
            };
            const float4* dptr = reinterpret_cast<const float4*>(a.data + img);
            const float4* sptr = reinterpret_cast<const float4*>(a.sigma + img);
            auto pass = [&]<bool MASKED>() {
              const uchar4* kptr = MASKED ? reinterpret_cast<const uchar4*>(a.mask + img) : nullptr;
#pragma unroll 4
              for (int idx = htid; idx < kGroups; idx += kHN) {
                const uint32_t p = px_addr(cut, idx / W4, (idx % W4) << 2);
                const float4 d4 = dptr[idx], s4 = sptr[idx];
                uchar4 k4 = make_uchar4(1, 1, 1, 1);
                if (MASKED) k4 = kptr[idx];
                uint4 m4 = lds128(p);
                if (UNCONV) add_unconv(m4, idx);
                uint4 gv;
                gv.x = __float_as_uint(one(__uint_as_float(m4.x), d4.x, s4.x, !MASKED || k4.x != 0));
                gv.y = __float_as_uint(one(__uint_as_float(m4.y), d4.y, s4.y, !MASKED || k4.y != 0));
                gv.z = __float_as_uint(one(__uint_as_float(m4.z), d4.z, s4.z, !MASKED || k4.z != 0));
                gv.w = __float_as_uint(one(__uint_as_float(m4.w), d4.w, s4.w, !MASKED || k4.w != 0));
                if (with_grad) {
                  sts128(p, gv);
                  if (UNCONV)                             // their gradient needs G itself, not PSF * G
                    *reinterpret_cast<float4*>(a.gseed + img + 4 * (size_t)idx) =
                        make_float4(__uint_as_float(gv.x), __uint_as_float(gv.y), __uint_as_float(gv.z), __uint_as_float(gv.w));
                }
              }
            };
            if (a.mask) pass.template operator()<true>();
            else pass.template operator()<false>();
          }
        }
        if (a.mode != 0) {
          chi2 = warp_sum(chi2);
          if (lane == 0) red[hw] = chi2;
          if (!isfinite(amax)) amax = 0.0f;                // a non-finite chi^2 is reported through chi2_part; keep the scale sane
          if (with_grad) inv_sc[s][g] = scale_and_split(cut, amax);     // its first barrier also publishes red[]
          else help_sync();
          if (htid == 0 && b >= 0) {
            float t = 0.0f;
            for (int w = 0; w < kHelp; ++w) t += red[w];
            a.chi2_part[b] = t;
          }
          help_sync();                                     // red[] may be rewritten
        }
      }
    };

    // a5: the partial sums of every component from A (slot, fp32)
    auto gradient = [&](int item, int s) {
#pragma unroll
      for (int g = 0; g < G; ++g) {
        const int b = galaxy(item, g);
        const uint32_t cut = cut_addr(s, g);
        for (int c = 0; c < a.md.n_comp; ++c) {
          float sm[kNSum];
#pragma unroll
          for (int k = 0; k < kNSum; ++k) sm[k] = 0.0f;
          if (b >= 0) {
            const CompConst cc = a.cc[(size_t)b * a.md.n_comp + c];
            const bool box = a.md.box[c] != 0, conv = !UNCONV || a.md.conv[c] != 0;
            dispatch_kind(a.md.kind[c], [&]<int KIND>() {
              GradAcc<KIND> acc;
              acc.init();
              for (int idx = htid; idx < kGroups; idx += kHN) {
                const int R = idx / W4, x = (idx % W4) << 2;
                float seed[4];
                if (conv) {                                // A = PSF * G, in the slot
                  const uint4 q = lds128(px_addr(cut, R, x));
                  seed[0] = __uint_as_float(q.x); seed[1] = __uint_as_float(q.y); seed[2] = __uint_as_float(q.z); seed[3] = __uint_as_float(q.w);
                } else {                                   // G itself (written by this CTA's residual pass)
                  const float4 q = __ldcg(reinterpret_cast<const float4*>(a.gseed + (size_t)b * SIDE * SIDE) + idx);
                  seed[0] = q.x; seed[1] = q.y; seed[2] = q.z; seed[3] = q.w;
                }
                if (box) {                                 // Eq. 2 with B != 0: per-pixel geometry
#pragma unroll
                  for (int k = 0; k < 4; ++k)
                    grad_accumulate<KIND>(cc, true, seed[k], (float)(x + k) + 0.5f, (float)SIDE - 0.5f - (float)R, sm);
                } else {
                  grad_add4<KIND>(acc, cc, seed, (float)x + 0.5f, (float)SIDE - 0.5f - (float)R);
                }
              }
              if (!box) { acc.finish(cc, sm); sm[8] = sm[2]; }
            });
          }
#pragma unroll
          for (int k = 0; k < kNSum; ++k) {
            const float v = warp_sum(sm[k]);
            if (lane == 0) red[hw * kNSum + k] = v;
          }
          help_sync();
          if (htid < kNSum && b >= 0) {
            float t = 0.0f;
            for (int w = 0; w < kHelp; ++w) t += red[w * kNSum + htid];
            a.grad_part[((size_t)b * a.md.n_comp + c) * kNSum + htid] = t;
          }
          help_sync();
        }
      }
    };

    auto feed = [&](int item, int s) { if (item < n_items) produce(item, s); };
    feed(0, 0);
    feed(1, 1);
    for (int m = 0; 2 * m < n_items; ++m) {
      for (int s = 0; s < 2; ++s) {                       // after C1: residual
        const int item = 2 * m + s;
        if (item >= n_items) continue;
        drain(item, s);
        tr.ev(TR_RESIDUAL, item);
        residual(item, s);
        if (with_grad) signal_input(s);                    // G is in place: the adjoint convolution may start
        tr.ev(TR_RESIDUAL_END, item);
        if (!with_grad) feed(item + 2, s);
      }
      if (with_grad) {
        for (int s = 0; s < 2; ++s) {                     // after C2: gradient, then the next cutouts
          const int item = 2 * m + s;
          if (item >= n_items) continue;
          drain(item, s);
          tr.ev(TR_GRADIENT, item);
          gradient(item, s);
          tr.ev(TR_GRADIENT_END, item);
          feed(item + 2, s);
        }
      }
    }
  } else if (wid < kLastWarp) {
    // ----------------------------------- MMA issue ------------------------------------
    // (the accumulator rows are template arguments so that every address of the issue loop is warp-uniform at
    // compile time and stays in uniform registers)
    static_assert(kMmaWarps == 4, "accumulator rows w, w + 4, ... per MMA warp");
    const uint32_t b0 = smem_u32(bars), r0 = smem_u32(ring);
    if (wid == 4 + kHelp) fused_mma_role<KP, 0, Gm::kRingF>(n_items, phases, b0, r0, tD, tA, a.trace);
    else if (wid == 5 + kHelp) fused_mma_role<KP, 1, Gm::kRingF>(n_items, phases, b0, r0, tD, tA);
    else if (wid == 6 + kHelp) fused_mma_role<KP, 2, Gm::kRingF>(n_items, phases, b0, r0, tD, tA);
    else fused_mma_role<KP, 3, Gm::kRingF>(n_items, phases, b0, r0, tD, tA);
  } else {
    // ------------------------------- tap-row producer --------------------------------
    // in the order of first use on its side: window row y = seq(i) brings tap row y (r = 0) on the low side and
    // tap row y - (kTileR - 1) on the high side.  Several cutouts per pass share one PSF (the host sees to it).
    if (lane == 0) {
      int jc = 0;
      for_each_job(n_items, phases, [&](int item, int ph, int) {
        const int b = galaxy(item, 0);
        const uint8_t* tab = (ph ? a.btab_adj : a.btab_fwd) + (size_t)(b >= 0 ? b : 0) * a.btab_stride;
        for (int i = 0; i < C::NY; ++i) {
          const int y = C::seq(i);
          const int ta = (i & 1) ? y - (kTileR - 1) : y;
          if ((i & 1) ? (ta < C::kNLow || ta >= KP) : (ta >= C::kNLow)) continue;
          const int slot = C::template slot_of<Gm::kRingF>(ta);
          const uint32_t gen = (uint32_t)(jc * C::template uses_of_slot<Gm::kRingF>(slot) + C::template index_in_slot<Gm::kRingF>(ta));
          mbar_wait(bar(F_B_EMPTY + slot), (gen & 1) ^ 1);
          mbar_expect_tx(bar(F_B_FULL + slot), C::kTapBytes);
          bulk_g2s(smem_u32(ring + (size_t)slot * C::kTapBytes), tab + (size_t)ta * C::kTapBytes, C::kTapBytes, bar(F_B_FULL + slot));
        }
        ++jc;
      });
    }
  }
  fence_before();
  __syncthreads();
  if (wid == kLastWarp) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tm) : "memory");
}

// ---------------------------------------------------------------------------------------------------
// Cutouts above 128 px: the same engine on SUPER-TILES of 128 lanes (128 x 128 or 64 x 256 pixels, whichever
// covers the cutout with the fewest), G through global memory between the forward and the backward kernel
// as in the FFMA2 tile kernels (k_forward / k_backward).  One shared-memory slot holds the super-tile plus
// its halo (two do not fit beside the tap-row rings), so an item's input is built while the tensor pipe
// idles; everything after the convolution, however, runs beside the NEXT item's convolution: the accumulators
// are double buffered in tensor memory and leave it through a 16 KB transposition buffer, never through the slot.
//   k_tc_tile<KP, TRB, false>  fill: a1 render S on tile + halo, scale, split | C1 | post: a3 residual, G to
//                              global, chi^2 partial (mode 0: M to global)
//   k_tc_tile<KP, TRB, true>   fill: G tile + halo from global, scale, split  | C2 | post: a5 partial sums
// Helper order: fill(0), fill(1) || post(0) ... : fill(n + 1) waits for the window-row warps to have staged the
// last row of item n (F_SLOT_FREE), post(n) for its last MMA (F_D_FULL).
// ---------------------------------------------------------------------------------------------------
struct TileTcArgs {
  ModelDesc md;
  int B, H, W;
  int tiles_x, tiles_y;      // super-tiles per cutout
  int mode;                  // forward kernel: 0 render (write M to out), 1 / 2 chi^2 (G to gbuf when 2)
  const CompConst* cc;
  const uint8_t* btab; long long btab_stride; const float* bscale;
  const float* data; const float* sigma; const uint8_t* mask;
  float* out;                // mode 0: model image
  float* gbuf;               // [B,H,W] back-seed G: written by the forward kernel, read by the backward kernel
  float* sbuf;               // forward kernel: [gridDim.x][kTileScratchFloats] scratch, S of a CTA's next item (L2 resident)
  float* chi2_part;          // [B, tiles]
  int any_unconv;            // the model has components that do not go through the PSF
  float* gmax_part;          // [B, tiles] largest |G| of a tile: forward kernel (mode 2) -> backward kernel
  float* grad_part;          // [B, tiles, n_comp, kNSum]
  const int* frozen; const int* live; const int* n_live;
  unsigned long long* trace; // gm_trace_set (CTA 0), or nullptr
};

constexpr int kTileMaxCtas = 160;            // the super-tile kernels launch at most this many CTAs (one per SM)
constexpr int kTileScratchFloats = 32768;    // >= (tile + halo) pixels of any super-tile: 104 x 296 at K = 41

template <int KP, int TRB> struct TileCfg {
  using C = Cfg<KP>;
  static constexpr int TCB = 128 / TRB;                       // tile columns of a super-tile
  static constexpr int TH = kTileR * TRB, TW = kTileC * TCB;  // pixels of a super-tile
  static constexpr int RR = TH + KP - 1;                      // slot rows: tile + halo
  static constexpr int RW = TW + KP - 1;                      // columns that carry data
  static constexpr int kPitchT = (TW - kTileC + 16 * C::NCH + 31) / 32 * 32;   // + window padding of the last tile column, whole swizzle groups
  static constexpr int kSlotWordsT = RR * kPitchT;
  // transposition buffer of the accumulators: all 128 columns of every lane (the whole tile, 64 KB) where that
  // leaves the tap-row rings at least 6 slots each (K = 25), else 32 columns at a time (16 KB, four rounds)
  static constexpr size_t kFixedBase = kAlignSlack + Roles<kTileHW>::kHeaderBytes + (size_t)kSlotWordsT * 4;
  static constexpr int kLdPerPiece = (kSmemLimit - kFixedBase - (size_t)C::kDCols * 128 * 4) / (2 * (size_t)C::kTapBytes) >= 6 ? C::kDCols / 32 : 1;
  static constexpr int kPieceWords = 128 * 32 * kLdPerPiece;
  static constexpr size_t kFixed = kFixedBase + (size_t)kPieceWords * 4;
  static constexpr int kRingT = ((kSmemLimit - kFixed) / (2 * (size_t)C::kTapBytes)) >= (size_t)kMaxRing
                                    ? kMaxRing : (int)((kSmemLimit - kFixed) / (2 * (size_t)C::kTapBytes));
  static_assert(kRingT >= kTileR + 1, "tap-row rings");
  static constexpr size_t kSmem = kFixed + (size_t)(2 * kRingT) * C::kTapBytes;
  static_assert(kSmem <= kSmemLimit, "shared memory");
  static_assert(TW % 32 == 0 && TW >= 32, "rows of the transposition buffer are whole swizzle groups");
  static_assert(RR * ((RW / 4) * 4) <= kTileScratchFloats, "scratch of the forward kernel");
};

template <int KP, int TRB, bool BWD, bool UNCONV>
__global__ void __launch_bounds__(Roles<kTileHW>::kThreads, 1) k_tc_tile(const TileTcArgs a) {
  using C = Cfg<KP>;
  using T = TileCfg<KP, TRB>;
  using Ro = Roles<kTileHW>;
  constexpr int h = C::h, kHN = Ro::kHN, kHelp = Ro::kHelp;
  extern __shared__ unsigned char smem_raw[];
  unsigned char* base = reinterpret_cast<unsigned char*>(((uintptr_t)smem_raw + (kAlignSlack - 1)) & ~(uintptr_t)(kAlignSlack - 1));
  uint64_t* bars = reinterpret_cast<uint64_t*>(base);
  uint32_t* tmem_base_s = reinterpret_cast<uint32_t*>(base + 512);
  float* red = reinterpret_cast<float*>(base + 528);
  float* redmax = red + kHelp * kNSum;
  unsigned char* ring = base + Ro::kHeaderBytes;
  uint32_t* slotw = reinterpret_cast<uint32_t*>(ring + (size_t)(2 * T::kRingT) * C::kTapBytes);
  uint32_t* piecew = slotw + T::kSlotWordsT;
  auto bar = [&](int i) -> uint32_t { return smem_u32(bars + i); };

  if ((long long)blockIdx.x >= (long long)(a.live ? *a.n_live : a.B) * a.tiles_x * a.tiles_y) return;   // no item for this CTA
  const int tid = threadIdx.x, wid = __shfl_sync(0xffffffffu, tid >> 5, 0), lane = tid & 31;
  if (tid == 0) {
    for (int i = 0; i < 2; ++i) { mbar_init(bar(F_IN_FULL + i), kHelp); mbar_init(bar(F_D_FULL + i), kMmaWarps); }
    for (int i = 0; i < kNBuf; ++i) { mbar_init(bar(F_A_FULL + i), 4); mbar_init(bar(F_A_EMPTY + i), kMmaWarps); }
    for (int i = 0; i < 2 * T::kRingT; ++i) { mbar_init(bar(F_B_FULL + i), 1); mbar_init(bar(F_B_EMPTY + i), kTileR); }
    mbar_init(bar(F_SLOT_FREE), 4);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  constexpr int kLastWarp = Ro::kLastWarp;
  if (wid == kLastWarp) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_base_s)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  for (int i = tid; i < T::kSlotWordsT; i += Ro::kThreads) slotw[i] = 0u;        // padding columns stay zero
  fence_before();
  __syncthreads();
  fence_after();
  const uint32_t tm = __shfl_sync(0xffffffffu, *tmem_base_s, 0);
  const uint32_t tD = tm, tA = tm + 2 * C::kDCols;
  const uint32_t slot = smem_u32(slotw), piece = smem_u32(piecew);

  // items of this CTA: (galaxy of the list, super-tile), entries blockIdx.x, + gridDim.x, ...
  const int tiles = a.tiles_x * a.tiles_y;
  const int n_gal = a.live ? *a.n_live : a.B;
  const int n_all = n_gal * tiles;
  const int n_items = (n_all - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
  auto item_of = [&](int it, int& b, int& tile) {
    const int e = (int)blockIdx.x + it * (int)gridDim.x;
    const int g = e / tiles;
    tile = e - g * tiles;
    b = a.live ? a.live[g] : g;
    if (a.frozen && a.frozen[b]) b = -1;
  };

  if (wid < 4) {
    // ------------------------- window rows -> tensor memory --------------------------
    const uint32_t lane_base = (uint32_t)(32 * wid) << 16;
    const int m = 32 * wid + lane, tr = m % TRB, tc = m / TRB;     // this lane's tile of the super-tile
    int row_count = 0;
    for (int it = 0; it < n_items; ++it) {
      const int s = it & 1;
      mbar_wait(bar(F_IN_FULL + s), (it >> 1) & 1);
      for (int i = 0; i < C::NY; ++i, ++row_count) {
        const int y = C::seq(i);
        const int buf = row_count % kNBuf;
        mbar_wait(bar(F_A_EMPTY + buf), ((row_count / kNBuf) & 1) ^ 1);
        fence_after();
        const int R = kTileR * tr + y;                             // slot row (row 0 = image row i0 - h)
        stage_window_row<KP>(slot + 4u * (uint32_t)(R * T::kPitchT), slot, true, (kTileC * tc) >> 2, T::kPitchT / 4, swz_of(R),
                             tA + (uint32_t)(buf * C::kACols) + lane_base);
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(F_A_FULL + buf));
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(F_SLOT_FREE));                 // every window row of the item is in tensor memory
    }
  } else if (wid < 4 + kHelp) {
    // ------------------------------------ helpers -------------------------------------
    const int hw = wid - 4, htid = tid - 128;
    const uint32_t lane_base = (uint32_t)(32 * (hw & 3)) << 16;
    auto px_addr = [&](int R, int c) -> uint32_t { return slot + 4u * (uint32_t)swz(R, c, T::kPitchT); };
    auto help_sync = [&]() { asm volatile("bar.sync 1, %0;" ::"n"(kHN) : "memory"); };
    constexpr int RW4 = T::RW / 4, kRegionGroups = T::RR * RW4;      // groups of four pixels of the tile + halo
    constexpr int TW4 = T::TW / 4;
    constexpr int kLdPP = T::kLdPerPiece;                                          // 32-column loads per piece
    constexpr int kPieceRows = kRowsPerLd * kLdPP * TRB, kPieceGroups = kPieceRows * TW4;   // a piece = 32 kLdPP accumulator columns of every tile
    constexpr int kPieces = C::kDCols / (32 * kLdPP);
    const float inv_rw4 = 1.0f / (float)RW4;
    float inv_sc[2] = {1.0f, 1.0f};
    Tracer tr;                                           // tags: TR_PRODUCE = fill / render ahead, TR_RESIDUAL / TR_GRADIENT = post
    tr.init(a.trace, TR_HELPER, htid == 0);

    // ---- forward kernel: S of item `it` on the tile + halo (zero outside the cutout) -> this CTA's scratch in global
    // memory (L2), as fp32.  Runs beside the convolution of item it - 1, so that the slot, the one thing the tensor
    // pipe waits for, is filled by a single load-scale-split pass.  Returns the largest magnitude (every thread the same).
    float* const scratch = BWD ? nullptr : a.sbuf + (size_t)blockIdx.x * kTileScratchFloats;
    auto render_ahead = [&](int it) -> float {
      int b, tile;
      item_of(it, b, tile);
      const int tile_y = tile / a.tiles_x, tile_x = tile - tile_y * a.tiles_x;
      const int i0 = tile_y * T::TH, j0 = tile_x * T::TW;          // tile origin in the cutout
      const CompConst* ccb = a.cc + (size_t)(b >= 0 ? b : 0) * a.md.n_comp;
      float amax = 0.0f;
      int c_first = -1, c_last = -1;                       // the components that go through the PSF
      for (int c = 0; c < a.md.n_comp; ++c)
        if (!UNCONV || a.md.conv[c]) { if (c_first < 0) c_first = c; c_last = c; }
      if (c_first < 0)                                     // none: S = 0
        for (int idx = htid; idx < kRegionGroups; idx += kHN) __stcg(reinterpret_cast<float4*>(scratch) + idx, make_float4(0.0f, 0.0f, 0.0f, 0.0f));
      for (int c = 0; c < a.md.n_comp; ++c) {
        if (UNCONV && !a.md.conv[c]) continue;
        const CompConst cc = ccb[c];
        const bool box = a.md.box[c] != 0;
        const bool first = c == c_first, last = c == c_last;
        dispatch_kind(a.md.kind[c], [&]<int KIND>() {
          for (int idx = htid; idx < kRegionGroups; idx += kHN) {
            const int R = (int)(((float)idx + 0.5f) * inv_rw4), x = (idx - R * RW4) << 2;
            const int i = i0 - h + R, j = j0 - h + x;
            float4* dst = reinterpret_cast<float4*>(scratch) + idx;
            float v[4] = {0.0f, 0.0f, 0.0f, 0.0f};
            if (b >= 0 && (unsigned)i < (unsigned)a.H && (unsigned)j < (unsigned)a.W) {        // W % 4 == 0: whole group in or out
              value4<KIND, kFastForward>(cc, box, (float)j + 0.5f, (float)a.H - 0.5f - (float)i, v);   // R:G1
              if (!first) {                                                  // this thread's own earlier store
                const float4 q = __ldcg(dst);
                v[0] += q.x; v[1] += q.y; v[2] += q.z; v[3] += q.w;
              }
              if (last) amax = fmaxf(fmaxf(amax, fmaxf(fabsf(v[0]), fabsf(v[1]))), fmaxf(fabsf(v[2]), fabsf(v[3])));
            }
            __stcg(dst, make_float4(v[0], v[1], v[2], v[3]));
          }
        });
      }
      if (!isfinite(amax)) amax = 0.0f;
      for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
      if (lane == 0) redmax[hw] = amax;
      help_sync();                                       // also: every store of the scratch is visible to the CTA
      float mx = redmax[0];
#pragma unroll
      for (int w = 1; w < kHelp; ++w) mx = fmaxf(mx, redmax[w]);
      help_sync();                                       // redmax may be rewritten
      return mx;
    };
    // scratch -> slot: scale by the power of two of `amax`, split into (hi, lo) halves; the input of item `it` is ready
    auto fill_from_scratch = [&](int it, float amax) {
      const float sc = pow2_scale(amax);
#pragma unroll 4
      for (int idx = htid; idx < kRegionGroups; idx += kHN) {
        const int R = (int)(((float)idx + 0.5f) * inv_rw4), x = (idx - R * RW4) << 2;
        const float4 v = __ldcg(reinterpret_cast<const float4*>(scratch) + idx);
        sts128(px_addr(R, x), make_uint4(split_pack(v.x * sc), split_pack(v.y * sc), split_pack(v.z * sc), split_pack(v.w * sc)));
      }
      inv_sc[it & 1] = 1.0f / sc;
      help_sync();                                       // the scratch may be rewritten (render_ahead of the next item)
      if (lane == 0) mbar_arrive(bar(F_IN_FULL + (it & 1)));
    };

    // ---- backward kernel: the slot of item `it`: G on the tile + halo from global memory, zero outside the cutout;
    // one pass: the scale comes from the tile maxima the forward kernel left (this tile and its neighbours)
    auto fill = [&](int it) {
      int b, tile;
      item_of(it, b, tile);
      const int tile_y = tile / a.tiles_x, tile_x = tile - tile_y * a.tiles_x;
      const int i0 = tile_y * T::TH, j0 = tile_x * T::TW;          // tile origin in the cutout
      const size_t img = (size_t)(b >= 0 ? b : 0) * a.H * a.W;
      float amax = 0.0f;
      if (b >= 0) {
        for (int ty = max(tile_y - 1, 0); ty <= min(tile_y + 1, a.tiles_y - 1); ++ty)
          for (int tx = max(tile_x - 1, 0); tx <= min(tile_x + 1, a.tiles_x - 1); ++tx)
            amax = fmaxf(amax, a.gmax_part[(size_t)b * tiles + ty * a.tiles_x + tx]);
      }
      if (!isfinite(amax)) amax = 0.0f;
      const float sc = pow2_scale(amax);
      const float* gsrc = a.gbuf + img;
#pragma unroll 4
      for (int idx = htid; idx < kRegionGroups; idx += kHN) {
        const int R = (int)(((float)idx + 0.5f) * inv_rw4), x = (idx - R * RW4) << 2;
        const int i = i0 - h + R, j = j0 - h + x;
        float4 v = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        if (b >= 0 && (unsigned)i < (unsigned)a.H && (unsigned)j < (unsigned)a.W) v = *reinterpret_cast<const float4*>(gsrc + (size_t)i * a.W + j);
        sts128(px_addr(R, x), make_uint4(split_pack(v.x * sc), split_pack(v.y * sc), split_pack(v.z * sc), split_pack(v.w * sc)));
      }
      inv_sc[it & 1] = 1.0f / sc;
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(F_IN_FULL + (it & 1)));
    };

    // accumulator columns 32 p .. 32 p + 31 of every lane -> the transposition buffer as a (kRowsPerLd TRB) x TW
    // sub-image: buffer row kRowsPerLd tr + rr = tile row tr, accumulator row kRowsPerLd p + rr; 16-byte chunks
    // XOR-swizzled with tr
    auto piece_in = [&](int s, int p, float inv) {
      const int g = hw >> 2;                               // one warp per lane quarter and load
      if (kLdPP > 1 || g == (p & 3)) {
        const int ld = kLdPP > 1 ? g : p;                  // which 32 columns of the lane
        const int m = 32 * (hw & 3) + lane, tr = m % TRB, tc = m / TRB;
        uint32_t v[32];
        tmem_ld32(tD + (uint32_t)(s * C::kDCols + 32 * ld) + lane_base, v);
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const int row = kRowsPerLd * kLdPP * tr + kRowsPerLd * (kLdPP > 1 ? ld : 0) + (4 * k) / kTileC;
          const int ch = (kTileC / 4) * tc + ((4 * k) % kTileC) / 4;
          sts128(piece + 4u * (uint32_t)(row * T::TW + ((ch ^ (tr & 7)) << 2)),
                 make_uint4(__float_as_uint(__uint_as_float(v[4 * k]) * inv), __float_as_uint(__uint_as_float(v[4 * k + 1]) * inv),
                            __float_as_uint(__uint_as_float(v[4 * k + 2]) * inv), __float_as_uint(__uint_as_float(v[4 * k + 3]) * inv)));
        }
      }
      help_sync();
    };
    // group idx of piece p: buffer address, and its pixel (R, x) of the tile
    auto piece_px = [&](int p, int idx, int& R, int& x) -> uint32_t {
      const int row = idx / TW4, ch = idx - row * TW4;
      const int tr = row / (kRowsPerLd * kLdPP);
      R = kTileR * tr + kRowsPerLd * kLdPP * p + (row - kRowsPerLd * kLdPP * tr);
      x = ch << 2;
      return piece + 4u * (uint32_t)(row * T::TW + ((ch ^ (tr & 7)) << 2));
    };

    // ---- everything after the convolution of item `it`, beside the convolution of item it + 1
    auto post = [&](int it) {
      const int s = it & 1;
      int b, tile;
      item_of(it, b, tile);
      const int tile_y = tile / a.tiles_x, tile_x = tile - tile_y * a.tiles_x;
      const int i0 = tile_y * T::TH, j0 = tile_x * T::TW;
      const size_t img = (size_t)(b >= 0 ? b : 0) * a.H * a.W;
      mbar_wait(bar(F_D_FULL + s), (it >> 1) & 1);
      fence_after();
      tr.ev(TR_JOB, it);                                   // the accumulators of the item are complete
      const float inv = inv_sc[s] * a.bscale[(a.btab_stride && b >= 0) ? b : 0];
      if (!BWD) {
        // a3 on the tile: residual, chi^2 partial, G to global (mode 0: M to global)
        float chi2 = 0.0f;
        auto one = [&](float mm, float d, float sg, bool used) -> float {
          float w = rcp_fast(sg * sg), rho = d - mm;
          w = used ? w : 0.0f;
          rho = used ? rho : 0.0f;
          const float t = w * rho;
          chi2 = fmaf(t, rho, chi2);
          return -2.0f * t;
        };
        float gmax = 0.0f;
        for (int p = 0; p < kPieces; ++p) {
          piece_in(s, p, inv);
          if (b >= 0) {
#pragma unroll 4
            for (int idx = htid; idx < kPieceGroups; idx += kHN) {
              int R, x;
              const uint32_t pa = piece_px(p, idx, R, x);
              const int i = i0 + R, j = j0 + x;
              if (i >= a.H || j >= a.W) continue;
              const size_t o = img + (size_t)i * a.W + j;
              uint4 m4 = lds128(pa);
              if (UNCONV) {                                // components that do not go through the PSF (R:C3)
                const CompConst* ccb = a.cc + (size_t)b * a.md.n_comp;
                const float y = (float)a.H - 0.5f - (float)i;
                float m[4] = {__uint_as_float(m4.x), __uint_as_float(m4.y), __uint_as_float(m4.z), __uint_as_float(m4.w)};
                for (int c = 0; c < a.md.n_comp; ++c) {
                  if (a.md.conv[c]) continue;
                  const CompConst cc = ccb[c];
                  const int kind = a.md.kind[c];
#pragma unroll
                  for (int k = 0; k < 4; ++k) {
                    const float U = (kind == GM_SKY) ? 1.0f : profile_value(kind, cc, geometry<false>(cc, a.md.box[c] != 0, (float)(j + k) + 0.5f, y).r);
                    m[k] = fmaf(cc.amp, U, m[k]);
                  }
                }
                m4 = make_uint4(__float_as_uint(m[0]), __float_as_uint(m[1]), __float_as_uint(m[2]), __float_as_uint(m[3]));
              }
              if (a.mode == 0) {
                *reinterpret_cast<float4*>(a.out + o) = make_float4(__uint_as_float(m4.x), __uint_as_float(m4.y), __uint_as_float(m4.z), __uint_as_float(m4.w));
              } else {
                const float4 d4 = *reinterpret_cast<const float4*>(a.data + o), s4 = *reinterpret_cast<const float4*>(a.sigma + o);
                uchar4 k4 = make_uchar4(1, 1, 1, 1);
                if (a.mask) k4 = *reinterpret_cast<const uchar4*>(a.mask + o);
                float4 g;
                g.x = one(__uint_as_float(m4.x), d4.x, s4.x, k4.x != 0);
                g.y = one(__uint_as_float(m4.y), d4.y, s4.y, k4.y != 0);
                g.z = one(__uint_as_float(m4.z), d4.z, s4.z, k4.z != 0);
                g.w = one(__uint_as_float(m4.w), d4.w, s4.w, k4.w != 0);
                gmax = fmaxf(fmaxf(gmax, fmaxf(fabsf(g.x), fabsf(g.y))), fmaxf(fabsf(g.z), fabsf(g.w)));
                if (a.mode == 2) *reinterpret_cast<float4*>(a.gbuf + o) = g;
              }
            }
          }
          help_sync();                                     // the buffer may be rewritten
        }
        if (a.mode != 0) {
          chi2 = warp_sum(chi2);
          for (int o2 = 16; o2 > 0; o2 >>= 1) gmax = fmaxf(gmax, __shfl_xor_sync(0xffffffffu, gmax, o2));
          if (lane == 0) { red[hw] = chi2; redmax[hw] = gmax; }
          help_sync();
          if (htid == 0 && b >= 0) {
            float t = 0.0f, mx = 0.0f;
            for (int w = 0; w < kHelp; ++w) { t += red[w]; mx = fmaxf(mx, redmax[w]); }
            a.chi2_part[(size_t)b * tiles + tile] = t;
            // the largest back-seed of the tile: the backward kernel scales its input by the maximum over the tile and
            // its neighbours, an upper bound of the maximum over tile + halo, and so needs no pass of its own for it
            if (a.mode == 2) a.gmax_part[(size_t)b * tiles + tile] = mx;
          }
          help_sync();
        }
      } else {
        // a5 on the tile: the partial sums of every component from A (the pieces are drained once per component)
        for (int c = 0; c < a.md.n_comp; ++c) {
          float sm[kNSum];
#pragma unroll
          for (int k = 0; k < kNSum; ++k) sm[k] = 0.0f;
          const CompConst cc = a.cc[(size_t)(b >= 0 ? b : 0) * a.md.n_comp + c];
          const bool box = a.md.box[c] != 0, conv = !UNCONV || a.md.conv[c] != 0;
          dispatch_kind(a.md.kind[c], [&]<int KIND>() {
            GradAcc<KIND> acc;
            acc.init();
            for (int p = 0; p < kPieces; ++p) {
              piece_in(s, p, inv);
              if (b >= 0) {
                for (int idx = htid; idx < kPieceGroups; idx += kHN) {
                  int R, x;
                  const uint32_t pa = piece_px(p, idx, R, x);
                  const int i = i0 + R, j = j0 + x;
                  if (i >= a.H || j >= a.W) continue;
                  float seed[4];
                  if (conv) {                                // A = PSF * G, from the accumulators
                    const uint4 q = lds128(pa);
                    seed[0] = __uint_as_float(q.x); seed[1] = __uint_as_float(q.y); seed[2] = __uint_as_float(q.z); seed[3] = __uint_as_float(q.w);
                  } else {                                   // G itself
                    const float4 q = *reinterpret_cast<const float4*>(a.gbuf + img + (size_t)i * a.W + j);
                    seed[0] = q.x; seed[1] = q.y; seed[2] = q.z; seed[3] = q.w;
                  }
                  if (box) {
#pragma unroll
                    for (int k = 0; k < 4; ++k)
                      grad_accumulate<KIND>(cc, true, seed[k], (float)(j + k) + 0.5f, (float)a.H - 0.5f - (float)i, sm);
                  } else {
                    grad_add4<KIND>(acc, cc, seed, (float)j + 0.5f, (float)a.H - 0.5f - (float)i);
                  }
                }
              }
              help_sync();
            }
            if (b >= 0 && !box) { acc.finish(cc, sm); sm[8] = sm[2]; }
          });
#pragma unroll
          for (int k = 0; k < kNSum; ++k) {
            const float v = warp_sum(sm[k]);
            if (lane == 0) red[hw * kNSum + k] = v;
          }
          help_sync();
          if (htid < kNSum && b >= 0) {
            float t = 0.0f;
            for (int w = 0; w < kHelp; ++w) t += red[w * kNSum + htid];
            a.grad_part[(((size_t)b * tiles + tile) * a.md.n_comp + c) * kNSum + htid] = t;
          }
          help_sync();
        }
      }
      fence_before();
    };

    if constexpr (!BWD) {
      float amax_next = n_items > 0 ? render_ahead(0) : 0.0f;
      for (int it = 0; it <= n_items; ++it) {
        if (it < n_items) {
          tr.ev(TR_DRAIN_WAIT, it);
          if (it > 0) mbar_wait(bar(F_SLOT_FREE), (it - 1) & 1);
          tr.ev(TR_DRAIN, it);
          fill_from_scratch(it, amax_next);                // the convolution of item `it` starts
          tr.ev(TR_PRODUCE_END, it);
        }
        if (it > 0) { tr.ev(TR_RESIDUAL, it - 1); post(it - 1); tr.ev(TR_RESIDUAL_END, it - 1); }
        if (it + 1 < n_items) { tr.ev(TR_PRODUCE, it + 1); amax_next = render_ahead(it + 1); }
      }
    } else {
      for (int it = 0; it <= n_items; ++it) {
        if (it < n_items) {
          tr.ev(TR_DRAIN_WAIT, it);
          if (it > 0) mbar_wait(bar(F_SLOT_FREE), (it - 1) & 1);
          tr.ev(TR_PRODUCE, it);
          fill(it);
          tr.ev(TR_PRODUCE_END, it);
        }
        if (it > 0) { tr.ev(TR_GRADIENT, it - 1); post(it - 1); tr.ev(TR_GRADIENT_END, it - 1); }
      }
    }
  } else if (wid < kLastWarp) {
    // ----------------------------------- MMA issue ------------------------------------
    const uint32_t b0 = smem_u32(bars), r0 = smem_u32(ring);
    if (wid == 4 + kHelp) fused_mma_role<KP, 0, T::kRingT>(n_items, 1, b0, r0, tD, tA, a.trace);
    else if (wid == 5 + kHelp) fused_mma_role<KP, 1, T::kRingT>(n_items, 1, b0, r0, tD, tA);
    else if (wid == 6 + kHelp) fused_mma_role<KP, 2, T::kRingT>(n_items, 1, b0, r0, tD, tA);
    else fused_mma_role<KP, 3, T::kRingT>(n_items, 1, b0, r0, tD, tA);
  } else {
    // ------------------------------- tap-row producer --------------------------------
    // (forward kernel: its idle lanes first ask the L2 for D, sigma and the mask of the item, which the residual
    // pass reads one convolution later: that pass waits on global memory)
    for (int it = 0; it < n_items; ++it) {
      if (!BWD && a.mode != 0) {
        int b, tile;
        item_of(it, b, tile);
        if (b >= 0) {
          const int tile_y = tile / a.tiles_x, tile_x = tile - tile_y * a.tiles_x;
          const int i0 = tile_y * T::TH, j0 = tile_x * T::TW;
          const size_t img = (size_t)b * a.H * a.W;
          constexpr int kLines = T::TW / 32;                       // 128-byte lines of floats per tile row
          for (int e = lane; e < T::TH * kLines; e += 32) {
            const int i = i0 + e / kLines, j = j0 + (e % kLines) * 32;
            if (i >= a.H || j >= a.W) continue;
            const size_t o = img + (size_t)i * a.W + j;
            asm volatile("prefetch.global.L2 [%0];" ::"l"(a.data + o));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(a.sigma + o));
            if (a.mask && (e % kLines) % 4 == 0) asm volatile("prefetch.global.L2 [%0];" ::"l"(a.mask + o));
          }
        }
      }
      if (BWD && it + 1 < n_items) {                        // backward kernel: G of the NEXT item's tile + halo
        int b, tile;
        item_of(it + 1, b, tile);
        if (b >= 0) {
          const int tile_y = tile / a.tiles_x, tile_x = tile - tile_y * a.tiles_x;
          const int i0 = tile_y * T::TH - h, j0 = tile_x * T::TW - h;
          const size_t img = (size_t)b * a.H * a.W;
          constexpr int kLines = (T::RW + 31) / 32 + 1;            // 128-byte lines that a row of the region may touch
          for (int e = lane; e < T::RR * kLines; e += 32) {
            const int i = i0 + e / kLines, j = ((j0 < 0 ? 0 : j0) & ~31) + (e % kLines) * 32;
            if ((unsigned)i >= (unsigned)a.H || j >= a.W || j > j0 + T::RW) continue;
            asm volatile("prefetch.global.L2 [%0];" ::"l"(a.gbuf + img + (size_t)i * a.W + j));
          }
        }
      }
      if (lane == 0) {
        int b, tile;
        item_of(it, b, tile);
        const uint8_t* tab = a.btab + (size_t)(b >= 0 ? b : 0) * a.btab_stride;
        for (int i = 0; i < C::NY; ++i) {
          const int y = C::seq(i);
          const int ta = (i & 1) ? y - (kTileR - 1) : y;
          if ((i & 1) ? (ta < C::kNLow || ta >= KP) : (ta >= C::kNLow)) continue;
          const int sl = C::template slot_of<T::kRingT>(ta);
          const uint32_t gen = (uint32_t)(it * C::template uses_of_slot<T::kRingT>(sl) + C::template index_in_slot<T::kRingT>(ta));
          mbar_wait(bar(F_B_EMPTY + sl), (gen & 1) ^ 1);
          mbar_expect_tx(bar(F_B_FULL + sl), C::kTapBytes);
          bulk_g2s(smem_u32(ring + (size_t)sl * C::kTapBytes), tab + (size_t)ta * C::kTapBytes, C::kTapBytes, bar(F_B_FULL + sl));
        }
      }
      __syncwarp();
    }
  }
  fence_before();
  __syncthreads();
  if (wid == kLastWarp) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tm) : "memory");
}

}  // namespace tc
}  // namespace gm
