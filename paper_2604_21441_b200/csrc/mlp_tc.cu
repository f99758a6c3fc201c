// mlp_tc.cu -- K5/K6 on the 5th-generation tensor cores: ONE persistent kernel runs, per 128-atom tile of one
// element, the whole per-element MLP forward (SURVEY.md Appendix A "Network") and its analytic backward to
// dE/dAEV (Appendix A "Backward"; eq. 2 needs dE/dr) without the activations ever leaving the SM:
//
//     F1  z1 = G  W1^T      F2  z2 = h1 W2^T      F3  z3 = h2 W3^T      (h = CELU(z + b), E_i = h3 . w4 + b4)
//     B3  d2 = dl3 W3       B2  d1 = dl2 W2       B1  g  = dl1 W1       (dl3 = w4 * c3, dl_l = d_l * c_l, c = CELU')
//
// Every GEMM is tcgen05.mma (kind::f16, M = 128, fp32 accumulators in TMEM) issued by one thread; the A operand
// (AEV tile, then each layer's activations / deltas) lives in shared memory in the canonical K-major
// SWIZZLE_128B layout and is rewritten in place by the epilogue warps; the B operand (weights) is streamed from
// L2 by the bulk-copy engine (cp.async.bulk, UBLKCP) through an mbarrier ring from images pre-tiled in exactly the
// shared-memory layout.  The operand is handed to the MMA warp panel by panel (64 columns), so a GEMM runs while the
// epilogue that feeds it is still at work; consecutive GEMMs alternate between two 256-column TMEM accumulators, and
// CELU' of layers 1-2 (packed to 16 bits) waits for the backward pass in a per-CTA, L2-resident global scratch.
//
// Arithmetic (NNP_MLP_F16X3): every operand x is split x = hi + lo with hi = fp16(x), lo = fp16(x - hi) and the
// product is hi*hi + lo*hi + hi*lo (three MMAs, fp32 accumulate): ~2^-21 relative operand error, i.e. fp32-grade
// (measured against the fp64 oracle in DESIGN.md).  NNP_MLP_F16X1 keeps only hi*hi.
#include <cuda_fp16.h>
#include <string.h>
#include <mutex>
#include <vector>
#include "nnp_internal.h"

namespace nnp {

// ------------------------------------------------------------------------------------------------ image geometry
// A B-operand matrix [N][K] (row n = output column, K contiguous) is cut into N-chunks of tc_chunk(N) rows
// (<= 256, one MMA each: every layer width of the supported networks is ONE chunk, so the A operand is read from
// shared memory once per k-step -- with two 128-row chunks the A re-read made the MMAs shared-memory bound) and
// K-panels of 64 columns.  Block (c, p) holds rows x 64 fp16 as rows x 128 bytes in
// the SWIZZLE_128B K-major layout (8-row atoms of 1024 B; 16-byte chunk index XOR row%8), hi half then lo half.
__host__ __device__ inline int tc_nchunks(int N) { return (N + 255) / 256; }
__host__ __device__ inline int tc_chunk(int N) { const int nc = tc_nchunks(N); return (((N + nc - 1) / nc) + 15) & ~15; }
__host__ __device__ inline int tc_npanels(int K) { return (K + 63) / 64; }
__host__ __device__ inline size_t tc_img_bytes(int N, int K) {
  return (size_t)tc_nchunks(N) * tc_npanels(K) * 2 * tc_chunk(N) * 128;
}
__host__ __device__ inline size_t tc_blk_off(int N, int K, int c, int p, int half) {
  return ((size_t)(c * tc_npanels(K) + p) * 2 + half) * tc_chunk(N) * 128;
}
__host__ __device__ inline int tc_elem_off(int r, int kk) {  // byte offset of element (row r, column kk < 64)
  return r * 128 + ((((kk >> 3) ^ (r & 7))) << 4) + (kk & 7) * 2;
}

struct TcNetImg { const uint8_t* w2; const uint8_t* w3; const uint8_t* w3t; const uint8_t* w2t; };
struct TcTable { TcNetImg n[MAX_S]; };

struct TcPackArgs { uint8_t* w1[MAX_S]; uint8_t* w1t[MAX_S]; };
struct TcPackAll { TcPackArgs m[MAX_MEMBERS]; };

struct TcModel {
  TcTable tab[MAX_MEMBERS];
  void* blob;
  NetTable* d_nets;        // device copy of the members' network tables
  TcTable* d_tabs;         // device copy of tab[]
};

struct TcWorkspace {
  uint8_t* w1img[MAX_MEMBERS][MAX_S];   // F1 image [N1][Kc] per member and slot (repacked when the column set changes)
  uint8_t* w1timg[MAX_MEMBERS][MAX_S];  // B1 image [Kc][N1]
  unsigned long long* key; // [2]: column-set key the images were packed for / scratch
  TcPackAll* d_pall;       // device copy of the layer-1 image pointer table
  int* done;               // [max_tiles] ensemble hand-over: members of a tile already accumulated (reset every call)
  uint32_t* cscr;          // [num_sms][TC_CSCR_WORDS] packed CELU' of the tile in flight, per CTA
  int num_sms;
  int smem_bytes[2];
};

// ------------------------------------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]^T, fp16 operands, fp32 accumulate, M = 128
__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
      "}\n" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc) : "memory");
}
// One k-step (K = 16) against a B half-block, issued by one elected lane of a CONVERGED warp (predicated, so the
// compiler emits straight-line code instead of a per-thread retry loop).  TWO = true: the B_hi block takes
// A_hi * B_hi and A_lo * B_hi; TWO = false: one product (A_hi * B_hi of the single-pass mode, or A_hi * B_lo).
template <bool TWO>
__device__ __forceinline__ void tc_mma_step(uint32_t d_tmem, uint64_t a0, uint64_t a1, uint64_t b, uint32_t idesc,
                                            uint32_t acc) {
  if (TWO) {
    asm volatile(
        "{\n"
        ".reg .pred pe, pa, pt;\n"
        "elect.sync _|pe, 0xffffffff;\n"
        "setp.ne.b32 pa, %5, 0;\n"
        "setp.eq.b32 pt, %5, %5;\n"
        "@pe tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %3, %4, pa;\n"
        "@pe tcgen05.mma.cta_group::1.kind::f16 [%0], %2, %3, %4, pt;\n"
        "}\n" ::"r"(d_tmem), "l"(a0), "l"(a1), "l"(b), "r"(idesc), "r"(acc) : "memory");
  } else {
    asm volatile(
        "{\n"
        ".reg .pred pe, pa;\n"
        "elect.sync _|pe, 0xffffffff;\n"
        "setp.ne.b32 pa, %4, 0;\n"
        "@pe tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, pa;\n"
        "}\n" ::"r"(d_tmem), "l"(a0), "l"(b), "r"(idesc), "r"(acc) : "memory");
  }
}
__device__ __forceinline__ void tc_commit_elect(uint32_t bar) {
  asm volatile(
      "{\n"
      ".reg .pred pe;\n"
      "elect.sync _|pe, 0xffffffff;\n"
      "@pe tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n"
      "}\n" ::"r"(bar) : "memory");
}
// K-major SWIZZLE_128B shared-memory matrix descriptor: start address >> 4, LBO (unused for swizzled K-major) = 1,
// SBO = 1024 B between 8-row atoms, descriptor version 1 (sm_100), layout type 2 = SWIZZLE_128B.
__device__ __forceinline__ uint64_t tc_desc(uint32_t saddr) {
  return (uint64_t)((saddr >> 4) & 0x3FFFu) | (1ull << 16) | (64ull << 32) | (1ull << 46) | (2ull << 61);
}
// instruction descriptor: D fp32 (bit 4), A/B fp16 (0), both K-major, N >> 3 at bit 17, M >> 4 at bit 24
__device__ __forceinline__ uint32_t tc_idesc(int N) { return (1u << 4) | ((uint32_t)(N >> 3) << 17) | (8u << 24); }

#define TC_R8(v, o) "=r"(v[o]), "=r"(v[o + 1]), "=r"(v[o + 2]), "=r"(v[o + 3]), "=r"(v[o + 4]), "=r"(v[o + 5]), "=r"(v[o + 6]), "=r"(v[o + 7])
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t* v) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : TC_R8(v, 0), TC_R8(v, 8) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void sts128(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ uint32_t h2_bits(__half2 h) { return *reinterpret_cast<uint32_t*>(&h); }
// (x0, x1) -> packed fp16 hi pair and lo pair (lo = fp16(x - hi))
__device__ __forceinline__ void split2(float x0, float x1, uint32_t& hi, uint32_t& lo) {
  const __half2 h = __floats2half2_rn(x0, x1);
  const float2 hf = __half22float2(h);
  hi = h2_bits(h);
  const float2 d = __ffma2_rn(hf, make_float2(-1.0f, -1.0f), make_float2(x0, x1));   // x - hi, exact, one packed instruction
  lo = h2_bits(__floats2half2_rn(d.x, d.y));
}
// ------------------------------------------------------------------------------------------------ layer-1 images
// The AEV columns that are materialised depend on the species present in the evaluation (GroupInfo::blkmap), so the
// layer-1 operand images are (re)packed on the device, only when that column set changed since the last call.

__device__ __forceinline__ void tc_store8(uint8_t* img, size_t blk_hi, size_t blk_lo, int r, int kk, const float* x) {
  uint32_t hi[4], lo[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) split2(x[2 * i], x[2 * i + 1], hi[i], lo[i]);
  const int eo = tc_elem_off(r, kk);
  *reinterpret_cast<uint4*>(img + blk_hi + eo) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
  *reinterpret_cast<uint4*>(img + blk_lo + eo) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
}

// L2 prefetch of [p, p + bytes) in 4 KB pieces, piece i by thread i of the `nthr` threads that share the range
__device__ __forceinline__ void tc_prefetch_l2(const uint8_t* p, size_t bytes, int i, int nthr) {
  for (size_t off = (size_t)i * 4096; off < bytes; off += (size_t)nthr * 4096) {
    const uint32_t sz = (uint32_t)min((size_t)4096, bytes - off) & ~15u;
    if (sz) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p + off), "r"(sz) : "memory");
  }
}

__global__ void __launch_bounds__(256)
k_tc_pack_w1(const NetTable* __restrict__ all_nets, const GroupInfo* __restrict__ grp, TcPackAll all,
             const TcTable* __restrict__ all_tabs, int kfull_all, unsigned long long* __restrict__ key, int* __restrict__ done,
             int max_tiles) {
  TL_SCOPE(0);
  pdl_trigger();
  {  // While the AEV kernel drains (this grid is resident ~10 us before its wait returns): pull the operand images of the
     // MLP kernel into L2.  After other work has gone through L2 (bench.py flushes it between steps) the first wave of
     // tiles otherwise streams its weights at DRAM latency, three 32 KB stages at a time.  Hints only: the images are static
     // model data (layer 1: as packed for the last column set); Kc may be read early here -- it only sizes a hint.
    const Net& pn = all_nets[blockIdx.z].net[blockIdx.y];
    if (kfull_all > 0 && pn.n_layers == 4) {   // (kfull_all = 0: stage profiling -- nothing to overlap with, no prefetch)
      const int N1 = pn.dims[1], N2 = pn.dims[2], N3 = pn.dims[3];
      const int kc = min(max(grp->Kc, 32), kfull_all) & ~31;
      const TcNetImg& im = all_tabs[blockIdx.z].n[blockIdx.y];
      const int i = blockIdx.x * blockDim.x + threadIdx.x, nthr = gridDim.x * blockDim.x;
      tc_prefetch_l2(all.m[blockIdx.z].w1[blockIdx.y], tc_img_bytes(N1, kc), i, nthr);
      tc_prefetch_l2(im.w2, tc_img_bytes(N2, N1), i, nthr);
      tc_prefetch_l2(im.w3, tc_img_bytes(N3, N2), i, nthr);
      tc_prefetch_l2(im.w3t, tc_img_bytes(N2, N3), i, nthr);
      tc_prefetch_l2(im.w2t, tc_img_bytes(N1, N2), i, nthr);
      tc_prefetch_l2(all.m[blockIdx.z].w1t[blockIdx.y], tc_img_bytes(kc, N1), i, nthr);
    }
  }
  pdl_wait();
  TL_WAITED(0);
  {  // every call: clear the ensemble hand-over flags of the MLP kernel that follows
    const int nthr = gridDim.x * gridDim.y * gridDim.z * blockDim.x;
    const int gid = ((blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x) * blockDim.x + threadIdx.x;
    for (int i = gid; i < max_tiles; i += nthr) done[i] = 0;
  }
  const unsigned long long want = grp->colkey;
  if (key[0] == want) return;
  if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && threadIdx.x == 0) key[1] = want;
  const int slot = blockIdx.y;
  const TcPackArgs& a = all.m[blockIdx.z];
  const Net& net = all_nets[blockIdx.z].net[slot];
  if (net.n_layers == 0 || grp->count[slot] == 0) return;
  const int Kc = grp->Kc, N1 = net.dims[1], Kfull = net.dims[0];
  const float* __restrict__ W1 = net.W[0];  // [N1][Kfull], internal column order
  const int nF = N1 * (Kc / 8), nB = Kc * (N1 / 8);
  for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < nF + nB; idx += gridDim.x * blockDim.x) {
    float x[8];
    if (idx < nF) {  // F1 image: B[n][k] = W1[n][col(k)]
      const int n = idx / (Kc / 8), k = (idx % (Kc / 8)) * 8;
      const float* src = W1 + (size_t)n * Kfull + grp->blkmap[k >> 5] * BLK + (k & 31);
#pragma unroll
      for (int i = 0; i < 8; ++i) x[i] = src[i];
      const int ch = tc_chunk(N1), c = n / ch, p = k >> 6;
      tc_store8(a.w1[slot], tc_blk_off(N1, Kc, c, p, 0), tc_blk_off(N1, Kc, c, p, 1), n - c * ch, k & 63, x);
    } else {         // B1 image: B[n][k] = W1[k][col(n)]
      const int i2 = idx - nF, n = i2 / (N1 / 8), k = (i2 % (N1 / 8)) * 8;
      const float* src = W1 + (size_t)k * Kfull + grp->blkmap[n >> 5] * BLK + (n & 31);
#pragma unroll
      for (int i = 0; i < 8; ++i) x[i] = src[(size_t)i * Kfull];
      const int ch = tc_chunk(Kc), c = n / ch, p = k >> 6;
      tc_store8(a.w1t[slot], tc_blk_off(Kc, N1, c, p, 0), tc_blk_off(Kc, N1, c, p, 1), n - c * ch, k & 63, x);
    }
  }
}

// ------------------------------------------------------------------------------------------------ the fused kernel
constexpr int TC_EPI_WARPS = 16;                      // loader / epilogue warps (four per TMEM lane quarter)
constexpr int TC_NPART = TC_EPI_WARPS / 4;            // warps sharing a lane quarter split the 16-column chunks
constexpr int TC_THREADS = (TC_EPI_WARPS + 2) * 32;   // + weight producer warp + MMA issuer warp
constexpr uint32_t TC_PANEL = 16384;                  // 128 rows x 128 B
constexpr uint32_t TC_LO = 4 * TC_PANEL;              // lo half of the A buffer
constexpr uint32_t TC_ACCW = 256;                     // TMEM: two 256-column accumulators (columns 0 and 256), used alternately
constexpr int TC_CW1 = 256, TC_CW2 = 256;             // words per row of CELU' (fp32) of layers 1 and 2 (global scratch)
constexpr int TC_CSCR_WORDS = (TC_CW1 + TC_CW2) * 128;  // per CTA: 256 KB, written in the forward and read back in the backward
                                                      // epilogues by the same thread; 38 MB for 148 CTAs, L2-resident

template <int NPASS> struct TcCfg {
  static constexpr int NH = (NPASS == 3) ? 2 : 1;
  static constexpr int NST = (NPASS == 3) ? 3 : 4;
  static constexpr uint32_t ABUF = NH * 4 * TC_PANEL;
  static constexpr uint32_t STAGE = 2 * TC_PANEL;               // one half-block: <= 256 rows x 128 B
  static constexpr uint32_t BARS = ABUF + NST * STAGE;          // full[NST], empty[NST], panel[4], acc_full
  static constexpr uint32_t TPTR = BARS + (2 * NST + 5) * 8;
  static constexpr uint32_t EPART = TPTR + 16;
  static constexpr uint32_t TOTAL = EPART + (TC_NPART - 1) * 128 * 4;
};

struct TileNet {
  int N1, N2, N3, Kc;
  const uint8_t *f1, *w2, *w3, *w3t, *w2t, *b1;
};

// The six GEMMs of one tile as "rounds": a round reads the A operand resident in shared memory (<= 4 K-panels) and
// fills <= 256 accumulator columns (one N-chunk).  F1 is K-streamed in rounds of 4 panels when Kc > 256, B1 is
// N-streamed in rounds of one chunk when Kc > 256.  A ring stage holds one half-block (hi or lo) of B.  The producer and the MMA issuer walk the same table with ONE
// copy of their block loop (an inlined copy per GEMM made the kernel overflow the instruction cache).
struct TcRound {
  const uint8_t* img;   // B image [N][K]
  int N, K, c0, c1, p0, p1, acc_first;
};
constexpr int TC_MAX_ROUNDS = 16;

__device__ __forceinline__ int tc_build_rounds(const TileNet& t, TcRound* r) {
  int n = 0;
  const int np = tc_npanels(t.Kc);
  for (int p0 = 0; p0 < np && n < TC_MAX_ROUNDS - 5; p0 += 4)
    r[n++] = TcRound{t.f1, t.N1, t.Kc, 0, tc_nchunks(t.N1), p0, min(np, p0 + 4), p0 > 0};
  r[n++] = TcRound{t.w2, t.N2, t.N1, 0, tc_nchunks(t.N2), 0, tc_npanels(t.N1), 0};
  r[n++] = TcRound{t.w3, t.N3, t.N2, 0, tc_nchunks(t.N3), 0, tc_npanels(t.N2), 0};
  r[n++] = TcRound{t.w3t, t.N2, t.N3, 0, tc_nchunks(t.N2), 0, tc_npanels(t.N3), 0};
  r[n++] = TcRound{t.w2t, t.N1, t.N2, 0, tc_nchunks(t.N1), 0, tc_npanels(t.N2), 0};
  const int nc = tc_nchunks(t.Kc);
  for (int c0 = 0; c0 < nc && n < TC_MAX_ROUNDS; ++c0)
    r[n++] = TcRound{t.b1, t.Kc, t.N1, c0, c0 + 1, 0, tc_npanels(t.N1), 0};
  return n;
}

template <int NPASS>
__device__ __forceinline__ void tc_store_act(uint32_t abuf, int row, int j, const uint32_t* hi, const uint32_t* lo) {
  // columns [16j, 16j+16) of `row` -> two 16-byte chunks of K-panel j/4 (conflict-free: chunk XOR row%8)
  const uint32_t base = abuf + (uint32_t)(j >> 2) * TC_PANEL + (uint32_t)row * 128u;
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    const uint32_t off = (uint32_t)((((j & 3) * 2 + i) ^ (row & 7)) << 4);
    sts128(base + off, hi[4 * i], hi[4 * i + 1], hi[4 * i + 2], hi[4 * i + 3]);
    if (NPASS == 3) sts128(base + TC_LO + off, lo[4 * i], lo[4 * i + 1], lo[4 * i + 2], lo[4 * i + 3]);
  }
}

// SM-clock timeline of CTA 0's first rounds (debug export nnp_debug_mlp_timeline): where a tile's time goes.  Profiling
// scaffolding: compiled in only with -DNNP_TC_TIMELINE (the product kernel carries no instrumentation).
#ifdef NNP_TC_TIMELINE
__device__ long long g_tc_timeline[64];
#define TC_STAMP() do { if (blockIdx.x == 0 && threadIdx.x == 0 && tl < 64) g_tc_timeline[tl++] = clock64(); } while (0)
#else
#define TC_STAMP() do { } while (0)
#endif

template <int NPASS>
__global__ void __launch_bounds__(TC_THREADS, 1)
k_mlp_tc(const NetTable* __restrict__ all_nets, const TcTable* __restrict__ all_tabs,
         const TcPackAll* __restrict__ w1all, const GroupInfo* __restrict__ grp,
         const TileInfo* __restrict__ tiles, const float* __restrict__ aev, float* __restrict__ daev,
         float* __restrict__ e_atom, unsigned long long* __restrict__ key, int* __restrict__ done, int n_members,
         float escale, uint32_t* cscr) {
  using C = TcCfg<NPASS>;
  extern __shared__ __align__(1024) uint8_t smem[];
  const uint32_t sbase = smem_u32(smem);
  const uint32_t abuf = sbase, stage0 = sbase + C::ABUF;
  const uint32_t bar_full = sbase + C::BARS, bar_empty = bar_full + 8 * C::NST;
  const uint32_t bar_panel = bar_empty + 8 * C::NST, bar_acc = bar_panel + 32;
  volatile uint32_t* tptr = reinterpret_cast<volatile uint32_t*>(smem + C::TPTR);
  float* e_part = reinterpret_cast<float*>(smem + C::EPART);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  TL_SCOPE(1);

  if (threadIdx.x == 0) {
    for (int i = 0; i < C::NST; ++i) { mbar_init(bar_full + 8 * i, 1); mbar_init(bar_empty + 8 * i, 1); }
    for (int i = 0; i < 4; ++i) mbar_init(bar_panel + 8 * i, TC_EPI_WARPS * 32);
    mbar_init(bar_acc, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == TC_EPI_WARPS + 1) {  // the MMA warp owns the TMEM allocation (all 512 columns; one CTA per SM)
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(sbase + C::TPTR), "r"(512u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tptr;
  // barriers and TMEM are set up while the previous kernels drain; nothing they produce is read before this wait.
  // The AEV backward kernel is this grid's programmatic dependent: it starts on the SMs this grid has left.
  pdl_wait();
  pdl_trigger();
  TL_WAITED(1);
  const int n_tiles = grp->n_tiles, Kc = grp->Kc;

  // Work items are (member, tile) pairs in member-major order, dealt round-robin to the resident CTAs: with an
  // ensemble the 8 x 188 items fill the SMs evenly instead of 8 launches of 1.27 waves each.  Members of one tile
  // accumulate into e_atom / dE/dAEV in member order: a CTA waits (done[tile] == member) before its first
  // read-modify-write; the awaited item has a smaller index, so it is already running on a resident CTA.
  const int n_items = n_tiles * n_members;
  auto tile_net = [&](int w, int& t, int& mem, TileInfo& ti, TileNet& tn) {
    mem = w / n_tiles; t = w - mem * n_tiles;   // n_items > 0 implies n_tiles > 0
    ti = tiles[t];
    const Net& net = all_nets[mem].net[ti.slot];
    tn.N1 = net.dims[1]; tn.N2 = net.dims[2]; tn.N3 = net.dims[3]; tn.Kc = Kc;
    tn.f1 = w1all->m[mem].w1[ti.slot]; tn.b1 = w1all->m[mem].w1t[ti.slot];
    const TcNetImg& im = all_tabs[mem].n[ti.slot];
    tn.w2 = im.w2; tn.w3 = im.w3; tn.w3t = im.w3t; tn.w2t = im.w2t;
  };

  if (warp == TC_EPI_WARPS) {
    // ===== weight producer: streams every B block of every round, in order, through the stage ring =====
    if (lane == 0) {
      int s = 0; uint32_t ph = 0;
      for (int w = blockIdx.x; w < n_items; w += gridDim.x) {
        int t, mem; TileInfo ti; TileNet tn; tile_net(w, t, mem, ti, tn);
        TcRound rd[TC_MAX_ROUNDS];
        const int nrd = tc_build_rounds(tn, rd);
#pragma unroll 1
        for (int ir = 0; ir < nrd; ++ir) {
          const uint8_t* img = rd[ir].img;
          const int N = rd[ir].N, K = rd[ir].K, c0 = rd[ir].c0, c1 = rd[ir].c1, p0 = rd[ir].p0, p1 = rd[ir].p1;
          const int ch = tc_chunk(N);
          for (int c = c0; c < c1; ++c) {
            const uint32_t bytes = (uint32_t)min(ch, N - c * ch) * 128u;
            for (int p = p0; p < p1; ++p) {
              // each half-block is a stage and goes out as four bulk copies: more requests in flight towards L2
              const uint32_t qb = bytes >> 2;
#pragma unroll
              for (int h = 0; h < C::NH; ++h) {
                mbar_wait(bar_empty + 8 * s, ph ^ 1);
                mbar_expect_tx(bar_full + 8 * s, bytes);
                const uint8_t* src = img + tc_blk_off(N, K, c, p, h);
                const uint32_t dst = stage0 + s * C::STAGE;
#pragma unroll
                for (int u = 0; u < 4; ++u) bulk_g2s(dst + u * qb, src + u * qb, qb, bar_full + 8 * s);
                if (++s == C::NST) { s = 0; ph ^= 1; }
              }
            }
          }
        }
      }
    }
  } else if (warp == TC_EPI_WARPS + 1) {
    // ===== MMA issuer: the warp stays converged, tcgen05 ops are predicated on one elected lane.  Descriptors are
    // built once per block and advanced by 32 B (+2 in the address field) per k-step: the issue loop must stay a
    // handful of instructions per MMA, or the single issuing warp, not the tensor core, paces the GEMM. =====
    {
      int s = 0; uint32_t ph = 0, pph = 0, buf = 1;
      for (int w = blockIdx.x; w < n_items; w += gridDim.x) {
        int t, mem; TileInfo ti; TileNet tn; tile_net(w, t, mem, ti, tn);
        TcRound rd[TC_MAX_ROUNDS];
        const int nrd = tc_build_rounds(tn, rd);
#pragma unroll 1
        for (int ir = 0; ir < nrd; ++ir) {
          const int N = rd[ir].N, K = rd[ir].K, c0 = rd[ir].c0, c1 = rd[ir].c1, p0 = rd[ir].p0, p1 = rd[ir].p1;
          const bool acc_first = rd[ir].acc_first != 0;
          if (!acc_first) buf ^= 1;               // a new accumulation takes the other accumulator
          const int ch = tc_chunk(N);
          for (int c = c0; c < c1; ++c) {
            const int rows = min(ch, N - c * ch);
            const uint32_t idesc = tc_idesc(rows), d = tmem + buf * TC_ACCW;
            for (int p = p0; p < p1; ++p) {
              // the previous epilogue hands the A operand over panel by panel (every panel barrier completes once a round)
              mbar_wait(bar_panel + 8 * (p - p0), pph);
              tc_fence_after();
              const int nks = min(4, (K - p * 64) >> 4);
              const uint32_t a0 = abuf + (uint32_t)(p - p0) * TC_PANEL;
              {   // B_hi block: A_hi * B_hi (+ A_lo * B_hi for the split)
                mbar_wait(bar_full + 8 * s, ph);
                tc_fence_after();
                uint64_t ah = tc_desc(a0), al = tc_desc(a0 + TC_LO), b = tc_desc(stage0 + s * C::STAGE);
                uint32_t acc = (acc_first || p > p0) ? 1u : 0u;
#pragma unroll
                for (int ks = 0; ks < 4; ++ks) {
                  if (ks < nks) {
                    tc_mma_step<NPASS == 3>(d, ah, al, b, idesc, acc);
                    acc = 1u; ah += 2; al += 2; b += 2;
                  }
                }
                tc_commit_elect(bar_empty + 8 * s);  // frees the stage when these MMAs have read it
                if (++s == C::NST) { s = 0; ph ^= 1; }
              }
              if (NPASS == 3) {   // B_lo block: A_hi * B_lo
                mbar_wait(bar_full + 8 * s, ph);
                tc_fence_after();
                uint64_t ah = tc_desc(a0), b = tc_desc(stage0 + s * C::STAGE);
#pragma unroll
                for (int ks = 0; ks < 4; ++ks) {
                  if (ks < nks) {
                    tc_mma_step<false>(d, ah, ah, b, idesc, 1u);
                    ah += 2; b += 2;
                  }
                }
                tc_commit_elect(bar_empty + 8 * s);
                if (++s == C::NST) { s = 0; ph ^= 1; }
              }
            }
          }
          tc_commit_elect(bar_acc);                // accumulator complete (and the A operand no longer read)
          pph ^= 1;
        }
      }
    }
  } else {
    // ===== loader / epilogue warps: thread <-> tile row (TMEM lane); the TC_NPART warps of a lane quarter take the
    // 16-column chunks round-robin =====
    const int q = warp & 3, part = warp >> 2, row = q * 32 + lane;
    const uint32_t tlane = tmem + ((uint32_t)(q * 32) << 16);
    uint32_t fph = 0, buf = 1;
#ifdef NNP_TC_TIMELINE
    int tl = 0;   // timeline slot (block 0, thread 0 only): even = operand handed to the MMA warp, odd = accumulator back
#endif
    // Hand-over protocol.  The A operand goes to the MMA warp PANEL BY PANEL (64 columns): every thread arrives once a
    // round on each of the four panel barriers, as soon as its share of the panel is in shared memory, so the MMAs of
    // the next GEMM start on panel 0 while this epilogue is still producing panels 1-3.  That GEMM accumulates into the
    // OTHER 256-column TMEM accumulator (the epilogue is still reading this one); CELU' therefore waits for the
    // backward pass in a per-CTA global scratch (L2-resident) instead of TMEM.
    auto arrive_panel = [&](int i) {
      tc_fence_before();
      fence_proxy_async();
      if (i == 3) TC_STAMP();
      mbar_arrive(bar_panel + 8 * i);
    };
    auto arrive_all = [&]() {
      tc_fence_before();
      fence_proxy_async();
      TC_STAMP();
#pragma unroll
      for (int i = 0; i < 4; ++i) mbar_arrive(bar_panel + 8 * i);
    };
    auto wait_acc = [&]() {
      // ONE thread polls the mbarrier; the other 511 sleep in a hardware named barrier.  (512 threads spinning on
      // try_wait flood the shared-memory pipe that feeds the tensor core's operand reads.)
      if (threadIdx.x == 0) mbar_wait(bar_acc, fph);
      fph ^= 1;
      asm volatile("bar.sync 2, %0;" ::"n"(TC_EPI_WARPS * 32) : "memory");
      tc_fence_after();
      TC_STAMP();
    };
    float* const cs1 = reinterpret_cast<float*>(cscr) + (size_t)blockIdx.x * TC_CSCR_WORDS;   // CELU' of layer 1: [piece = column / 4][128 rows][4 floats]
    float* const cs2 = cs1 + TC_CW1 * 128;
    for (int w = blockIdx.x; w < n_items; w += gridDim.x) {
      int t, mem; TileInfo ti; TileNet tn; tile_net(w, t, mem, ti, tn);
      const Net& net = all_nets[mem].net[ti.slot];
      const bool accumulate = mem > 0;
      const float alpha = net.alpha, kexp = 1.4426950408889634f / alpha;
      const float2 alpha2 = make_float2(alpha, alpha), nalpha2 = make_float2(-alpha, -alpha), kexp2 = make_float2(kexp, kexp);
      const bool valid = row < ti.nvalid;
      // ---- F1 rounds: AEV columns [64 p0, 64 p1) -> fp16 hi/lo panels
      const int np = tc_npanels(Kc);
      for (int p0 = 0; p0 < np; p0 += 4) {
        const int k0 = p0 * 64, kw = min(Kc, k0 + 256) - k0, n16 = kw >> 3;
        constexpr int NT = TC_EPI_WARPS * 32;
        static_assert(NT == 512, "two batches of two 1024-item panels");
        // panel-major: a 64-column panel is 128 rows x 8 chunks of 8 floats = 1024 items, two per thread; a batch of two
        // panels keeps four loads per thread in flight, and each panel is handed to the MMA warp as soon as it is in place
#pragma unroll 1
        for (int pb = 0; pb < 4; pb += 2) {
          float4 x0[4], x1[4];
#pragma unroll
          for (int u = 0; u < 4; ++u) {   // all loads of the batch in flight before the first use
            const int within = (int)threadIdx.x + (u & 1) * NT, r = within >> 3, chn = (pb + (u >> 1)) * 8 + (within & 7);
            x0[u] = make_float4(0.f, 0.f, 0.f, 0.f); x1[u] = x0[u];
            if (chn < n16 && r < ti.nvalid) {
              const float4* src = reinterpret_cast<const float4*>(aev + (size_t)(ti.row0 + r) * Kc + k0 + chn * 8);
              x0[u] = __ldg(src); x1[u] = __ldg(src + 1);
            }
          }
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int within = (int)threadIdx.x + (u & 1) * NT, r = within >> 3, chn = (pb + (u >> 1)) * 8 + (within & 7);
            if (chn < n16) {
              uint32_t hi[4], lo[4];
              split2(x0[u].x, x0[u].y, hi[0], lo[0]); split2(x0[u].z, x0[u].w, hi[1], lo[1]);
              split2(x1[u].x, x1[u].y, hi[2], lo[2]); split2(x1[u].z, x1[u].w, hi[3], lo[3]);
              const uint32_t dst = abuf + (uint32_t)(chn >> 3) * TC_PANEL + (uint32_t)r * 128u + (uint32_t)(((chn & 7) ^ (r & 7)) << 4);
              sts128(dst, hi[0], hi[1], hi[2], hi[3]);
              if (NPASS == 3) sts128(dst + TC_LO, lo[0], lo[1], lo[2], lo[3]);
            }
            if (u & 1) arrive_panel(pb + (u >> 1));
          }
        }
        if (p0 == 0) buf ^= 1;   // mirrors the MMA warp: a new accumulation takes the other accumulator
        wait_acc();
      }
      // ---- forward hidden layers 1, 2: h = CELU(z + b) -> A operand of the next layer; CELU' packed to the scratch
#pragma unroll 1
      for (int l = 1; l <= 2; ++l) {
        const int N = (l == 1) ? tn.N1 : tn.N2;
        const float4* __restrict__ bias4 = reinterpret_cast<const float4*>(net.b[l - 1]);
        float* const cs = (l == 1) ? cs1 : cs2;
        const uint32_t tacc = tlane + buf * TC_ACCW;
#pragma unroll 1
        for (int pi4 = 0; pi4 < 4; ++pi4) {
          const int j = part + TC_NPART * pi4;
          if (j * 16 < N) {
          uint32_t v[16], hi[8], lo[8];
          float ce[16];
          tmem_ld16(tacc + j * 16, v);
          float4 bv[4];
#pragma unroll
          for (int i = 0; i < 4; ++i) bv[i] = __ldg(bias4 + j * 4 + i);
          tmem_wait_ld();
#pragma unroll
          for (int i = 0; i < 16; i += 2) {
            // CELU and CELU' of two columns in packed fp32: e = exp(min(z, 0) / alpha) = CELU'(z) (ex2(0) = 1 exactly, no
            // select), CELU(z) = max(z, 0) + alpha (e - 1) = fma(alpha, e, max(z, 0) - alpha)
            const float4 b4 = bv[i >> 2];
            const float2 z = __fadd2_rn(make_float2(__uint_as_float(v[i]), __uint_as_float(v[i + 1])),
                                        (i & 2) ? make_float2(b4.z, b4.w) : make_float2(b4.x, b4.y));
            const float2 t = __fmul2_rn(make_float2(fminf(z.x, 0.f), fminf(z.y, 0.f)), kexp2);
            const float2 e = make_float2(exp2f(t.x), exp2f(t.y));
            const float2 h = __ffma2_rn(alpha2, e, __fadd2_rn(make_float2(fmaxf(z.x, 0.f), fmaxf(z.y, 0.f)), nalpha2));
            ce[i] = e.x; ce[i + 1] = e.y;
            split2(h.x, h.y, hi[i >> 1], lo[i >> 1]);
          }
#pragma unroll
          for (int i = 0; i < 4; ++i)   // CELU' in fp32, piece-major like dE/dAEV: 512 contiguous bytes per warp store
            __stcg(reinterpret_cast<float4*>(cs + ((size_t)(4 * j + i) * 128 + row) * 4), make_float4(ce[4 * i], ce[4 * i + 1], ce[4 * i + 2], ce[4 * i + 3]));
          tc_store_act<NPASS>(abuf, row, j, hi, lo);
          }
          arrive_panel(pi4);
        }
        buf ^= 1;
        wait_acc();
      }
      // ---- layer 3 + output layer: E_i = h3 . w4 + b4;  dl3 = w4 * CELU'(z3) -> A operand of B3
      {
        const int nl = net.n_layers;
        const float4* __restrict__ bias4 = reinterpret_cast<const float4*>(net.b[2]);
        const float4* __restrict__ w44 = reinterpret_cast<const float4*>(net.W[nl - 1]);
        float2 e2 = make_float2(0.f, 0.f);
        const float2 esc2 = make_float2(escale, escale);
        const uint32_t tacc = tlane + buf * TC_ACCW;
#pragma unroll 1
        for (int pi4 = 0; pi4 < 4; ++pi4) {
          const int j = part + TC_NPART * pi4;
          if (j * 16 < tn.N3) {
          uint32_t v[16], hi[8], lo[8];
          tmem_ld16(tacc + j * 16, v);
          float4 bv[4], wv[4];
#pragma unroll
          for (int i = 0; i < 4; ++i) { bv[i] = __ldg(bias4 + j * 4 + i); wv[i] = __ldg(w44 + j * 4 + i); }
          tmem_wait_ld();
#pragma unroll
          for (int i = 0; i < 16; i += 2) {
            const float4 b4 = bv[i >> 2], w4 = wv[i >> 2];
            const float2 z = __fadd2_rn(make_float2(__uint_as_float(v[i]), __uint_as_float(v[i + 1])),
                                        (i & 2) ? make_float2(b4.z, b4.w) : make_float2(b4.x, b4.y));
            const float2 w2 = (i & 2) ? make_float2(w4.z, w4.w) : make_float2(w4.x, w4.y);   // escale = 1/members rides on dl3
            const float2 t = __fmul2_rn(make_float2(fminf(z.x, 0.f), fminf(z.y, 0.f)), kexp2);
            const float2 ce = make_float2(exp2f(t.x), exp2f(t.y));                            // CELU'(z) (1 for z > 0)
            const float2 h = __ffma2_rn(alpha2, ce, __fadd2_rn(make_float2(fmaxf(z.x, 0.f), fmaxf(z.y, 0.f)), nalpha2));
            e2 = __ffma2_rn(h, w2, e2);
            const float2 d = __fmul2_rn(__fmul2_rn(esc2, w2), ce);
            split2(d.x, d.y, hi[i >> 1], lo[i >> 1]);
          }
          tc_store_act<NPASS>(abuf, row, j, hi, lo);
          }
          arrive_panel(pi4);
        }
        float e = e2.x + e2.y;
        if (part > 0) e_part[(part - 1) * 128 + row] = e;
        if (accumulate && threadIdx.x == 0) {   // the previous member of this tile must have finished its updates
          int seen;
          do {
            asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(seen) : "l"(done + t) : "memory");
            if (seen < mem) __nanosleep(100);
          } while (seen < mem);
        }
        asm volatile("bar.sync 1, %0;" ::"n"(TC_EPI_WARPS * 32) : "memory");
        if (part == 0) {
#pragma unroll
          for (int pp = 0; pp < TC_NPART - 1; ++pp) e += e_part[pp * 128 + row];   // fixed order
          const float ev = valid ? escale * (e + __ldg(net.b[nl - 1])) : 0.f;
          e_atom[ti.row0 + row] = accumulate ? e_atom[ti.row0 + row] + ev : ev;   // ensemble: mean over members
        }
        buf ^= 1;   // (the wait for B3 sits at the top of the backward loop, behind the CELU' prefetch)
      }
      // ---- backward through layers 2, 1: dl_l = d_l * CELU'(z_l) -> A operand of the next backward GEMM.  The packed
      // CELU' words come back from the scratch one chunk ahead of their use (the first ones while the GEMM still runs).
#pragma unroll 1
      for (int l = 2; l >= 1; --l) {
        const int N = (l == 1) ? tn.N1 : tn.N2;
        const float* const cs = (l == 1) ? cs1 : cs2;
        float4 cn[4];   // this thread wrote these words itself in the forward pass
#pragma unroll
        for (int i = 0; i < 4; ++i)
          cn[i] = (part * 16 < N) ? __ldcg(reinterpret_cast<const float4*>(cs + ((size_t)(4 * part + i) * 128 + row) * 4)) : make_float4(0.f, 0.f, 0.f, 0.f);
        wait_acc();   // B3 (l = 2) / B2 (l = 1) complete
        const uint32_t tacc = tlane + buf * TC_ACCW;
#pragma unroll 1
        for (int pi4 = 0; pi4 < 4; ++pi4) {
          const int j = part + TC_NPART * pi4;
          if (j * 16 < N) {
          uint32_t v[16], hi[8], lo[8];
          tmem_ld16(tacc + j * 16, v);
          const float4 cc[4] = {cn[0], cn[1], cn[2], cn[3]};
          if ((j + TC_NPART) * 16 < N) {
#pragma unroll
            for (int i = 0; i < 4; ++i)
              cn[i] = __ldcg(reinterpret_cast<const float4*>(cs + ((size_t)(4 * (j + TC_NPART) + i) * 128 + row) * 4));
          }
          tmem_wait_ld();
#pragma unroll
          for (int i = 0; i < 16; i += 2) {
            const float4 c4 = cc[i >> 2];
            const float2 d = __fmul2_rn(make_float2(__uint_as_float(v[i]), __uint_as_float(v[i + 1])),
                                        (i & 2) ? make_float2(c4.z, c4.w) : make_float2(c4.x, c4.y));
            split2(d.x, d.y, hi[i >> 1], lo[i >> 1]);
          }
          tc_store_act<NPASS>(abuf, row, j, hi, lo);
          }
          arrive_panel(pi4);
        }
        buf ^= 1;
      }
      wait_acc();   // B1, first column chunk
      // ---- B1 rounds: g = dE/dAEV columns [n0, n0 + ncols) -> global (fp32, compacted AEV column order)
      {
        const int nc = tc_nchunks(Kc), ch = tc_chunk(Kc);
        for (int c0 = 0; c0 < nc; ++c0) {
          const int n0 = c0 * ch, ncols = min(Kc, (c0 + 1) * ch) - n0;
          float* __restrict__ dst = daev + daev_off((size_t)(ti.row0 + row), n0, Kc);   // piece-major tile layout
          const uint32_t tacc = tlane + buf * TC_ACCW;
          // the A operand (dl1) is unchanged: the MMAs of the next column chunk start now, into the other accumulator
          if (c0 + 1 < nc) { arrive_all(); buf ^= 1; }
#pragma unroll 1
          for (int j = part; j * 16 < ncols; j += TC_NPART) {
            uint32_t v[16];
            tmem_ld16(tacc + j * 16, v);
            tmem_wait_ld();
            if (valid) {
#pragma unroll
              for (int i = 0; i < 16; i += 4) {
                float4* o = reinterpret_cast<float4*>(dst + (size_t)(j * 4 + (i >> 2)) * (4 * TILE_M));
                float4 g = make_float4(__uint_as_float(v[i]), __uint_as_float(v[i + 1]), __uint_as_float(v[i + 2]), __uint_as_float(v[i + 3]));
                if (accumulate) { const float4 p = *o; g.x += p.x; g.y += p.y; g.z += p.z; g.w += p.w; }   // sum over members
                *o = g;
              }
            }
          }
          if (c0 + 1 < nc) wait_acc();
        }
        // the next tile's first round re-arms the panel barriers after its own loads (program order: the reads above are done)
        {   // publish this member's updates of the tile: to the CTA that holds the next member, and (last member) to
            // the AEV backward kernel, whose warps wait for their tile's flag
          __threadfence();
          asm volatile("bar.sync 2, %0;" ::"n"(TC_EPI_WARPS * 32) : "memory");
          if (threadIdx.x == 0) asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(done + t), "r"(mem + 1) : "memory");
          if (w == (int)blockIdx.x) TL_MARK(1);   // end of the CTA's first work item: first / last = the first wave's spread
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (blockIdx.x == 0 && threadIdx.x == 0) key[0] = key[1];
  if (warp == TC_EPI_WARPS + 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
  }
}

// ------------------------------------------------------------------------------------------------ host side
namespace {
void host_split(float x, uint16_t& hi, uint16_t& lo) {
  const __half h = __float2half_rn(x);
  const __half l = __float2half_rn(x - __half2float(h));
  memcpy(&hi, &h, 2); memcpy(&lo, &l, 2);
}
// image of B[n][k] = get(n, k), n < N, k < K
template <class G>
void host_image(std::vector<uint8_t>& blob, size_t base, int N, int K, G get) {
  const int ch = tc_chunk(N);
  for (int n = 0; n < N; ++n)
    for (int k = 0; k < K; ++k) {
      uint16_t hi, lo;
      host_split(get(n, k), hi, lo);
      const int c = n / ch, p = k >> 6, eo = tc_elem_off(n - c * ch, k & 63);
      memcpy(&blob[base + tc_blk_off(N, K, c, p, 0) + eo], &hi, 2);
      memcpy(&blob[base + tc_blk_off(N, K, c, p, 1) + eo], &lo, 2);
    }
}
bool tc_shape_ok(const nnp_mlp_desc& d) {
  if (d.n_layers != 4) return false;
  for (int l = 1; l <= 3; ++l)
    if (d.dims[l] % 32 || d.dims[l] < 32 || d.dims[l] > 256) return false;
  for (int l = 0; l < 4; ++l)
    for (size_t i = 0; i < (size_t)d.dims[l] * d.dims[l + 1]; ++i)
      if (!(fabsf(d.W[l][i]) < 6.0e4f)) return false;  // fp16 range of the hi part
  return true;
}
}  // namespace

int tc_model_create(nnp_model* m, const nnp_mlp_desc* nets /* [n_members][S] */) {
  m->tc = nullptr;
  const int S = m->aev.S, M = m->n_members;
  size_t total = 0;
  size_t off[MAX_MEMBERS][MAX_S][4];
  for (int mem = 0; mem < M; ++mem)
    for (int s = 0; s < S; ++s) {
      const nnp_mlp_desc& d = nets[(size_t)mem * S + s];
      if (d.n_layers == 0) continue;
      if (!tc_shape_ok(d)) return NNP_OK;  // no tensor-core image: workspaces stay in NNP_MLP_FP32_SIMT
      const int N1 = d.dims[1], N2 = d.dims[2], N3 = d.dims[3];
      const size_t sz[4] = {tc_img_bytes(N2, N1), tc_img_bytes(N3, N2), tc_img_bytes(N2, N3), tc_img_bytes(N1, N2)};
      for (int i = 0; i < 4; ++i) { off[mem][s][i] = total; total += (sz[i] + 1023) & ~(size_t)1023; }
    }
  std::vector<uint8_t> blob(total, 0);
  for (int mem = 0; mem < M; ++mem)
    for (int s = 0; s < S; ++s) {
      const nnp_mlp_desc& d = nets[(size_t)mem * S + s];
      if (d.n_layers == 0) continue;
      const int N1 = d.dims[1], N2 = d.dims[2], N3 = d.dims[3];
      const float *W2 = d.W[1], *W3 = d.W[2];  // [out][in]
      host_image(blob, off[mem][s][0], N2, N1, [&](int n, int k) { return W2[(size_t)n * N1 + k]; });  // F2: B = W2
      host_image(blob, off[mem][s][1], N3, N2, [&](int n, int k) { return W3[(size_t)n * N2 + k]; });  // F3: B = W3
      host_image(blob, off[mem][s][2], N2, N3, [&](int n, int k) { return W3[(size_t)k * N2 + n]; });  // B3: B = W3^T
      host_image(blob, off[mem][s][3], N1, N2, [&](int n, int k) { return W2[(size_t)k * N1 + n]; });  // B2: B = W2^T
    }
  TcModel* tm = new (std::nothrow) TcModel();
  if (!tm) return NNP_ERR_CUDA;
  memset(tm, 0, sizeof(*tm));
  if (cudaMalloc(&tm->blob, std::max<size_t>(total, 1024)) != cudaSuccess ||
      cudaMemcpy(tm->blob, blob.data(), total, cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMalloc(&tm->d_nets, sizeof(NetTable) * MAX_MEMBERS) != cudaSuccess ||
      cudaMemcpy(tm->d_nets, m->nets, sizeof(NetTable) * MAX_MEMBERS, cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMalloc(&tm->d_tabs, sizeof(TcTable) * MAX_MEMBERS) != cudaSuccess) {
    cudaGetLastError();
    if (tm->blob) cudaFree(tm->blob);
    if (tm->d_nets) cudaFree(tm->d_nets);
    if (tm->d_tabs) cudaFree(tm->d_tabs);
    delete tm;
    return NNP_ERR_CUDA;
  }
  for (int mem = 0; mem < M; ++mem)
    for (int s = 0; s < S; ++s) {
      if (nets[(size_t)mem * S + s].n_layers == 0) continue;
      const uint8_t* b = static_cast<const uint8_t*>(tm->blob);
      tm->tab[mem].n[s] = TcNetImg{b + off[mem][s][0], b + off[mem][s][1], b + off[mem][s][2], b + off[mem][s][3]};
    }
  if (cudaMemcpy(tm->d_tabs, tm->tab, sizeof(TcTable) * MAX_MEMBERS, cudaMemcpyHostToDevice) != cudaSuccess) {
    cudaGetLastError();
    cudaFree(tm->blob); cudaFree(tm->d_nets); cudaFree(tm->d_tabs);
    delete tm;
    return NNP_ERR_CUDA;
  }
  m->tc = tm;
  return NNP_OK;
}

void tc_model_destroy(nnp_model* m) {
  TcModel* tm = static_cast<TcModel*>(m->tc);
  if (!tm) return;
  if (tm->blob) cudaFree(tm->blob);
  if (tm->d_nets) cudaFree(tm->d_nets);
  if (tm->d_tabs) cudaFree(tm->d_tabs);
  delete tm;
  m->tc = nullptr;
}

int tc_workspace_create(nnp_workspace* ws) {
  ws->tc_ws = nullptr;
  const nnp_model* m = ws->model;
  if (!m->tc) return NNP_OK;
  TcWorkspace* tw = new (std::nothrow) TcWorkspace();
  if (!tw) return NNP_ERR_CUDA;
  memset(tw, 0, sizeof(*tw));
  ws->tc_ws = tw;
  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return NNP_ERR_CUDA;
  tw->num_sms = prop.multiProcessorCount;
  tw->smem_bytes[0] = (int)TcCfg<3>::TOTAL;
  tw->smem_bytes[1] = (int)TcCfg<1>::TOTAL;
  if (cudaFuncSetAttribute(k_mlp_tc<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, tw->smem_bytes[0]) != cudaSuccess ||
      cudaFuncSetAttribute(k_mlp_tc<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, tw->smem_bytes[1]) != cudaSuccess)
    return NNP_ERR_CUDA;
  for (int mem = 0; mem < m->n_members; ++mem)
    for (int s = 0; s < m->aev.S; ++s) {
      const Net& n = m->nets[mem].net[s];
      if (n.n_layers == 0) continue;
      const size_t b1 = tc_img_bytes(n.dims[1], m->Kfull), b2 = tc_img_bytes(m->Kfull, n.dims[1]);
      if (cudaMalloc(&tw->w1img[mem][s], b1) != cudaSuccess || cudaMalloc(&tw->w1timg[mem][s], b2) != cudaSuccess) return NNP_ERR_CUDA;
      cudaMemset(tw->w1img[mem][s], 0, b1);
      cudaMemset(tw->w1timg[mem][s], 0, b2);
    }
  if (cudaMalloc(&tw->key, 2 * sizeof(unsigned long long)) != cudaSuccess) return NNP_ERR_CUDA;
  cudaMemset(tw->key, 0, 2 * sizeof(unsigned long long));
  TcPackAll pall;
  memset(&pall, 0, sizeof(pall));
  for (int mem = 0; mem < MAX_MEMBERS; ++mem)
    for (int s = 0; s < MAX_S; ++s) { pall.m[mem].w1[s] = tw->w1img[mem][s]; pall.m[mem].w1t[s] = tw->w1timg[mem][s]; }
  if (cudaMalloc(&tw->d_pall, sizeof(TcPackAll)) != cudaSuccess ||
      cudaMemcpy(tw->d_pall, &pall, sizeof(TcPackAll), cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMalloc(&tw->done, sizeof(int) * (size_t)std::max(ws->max_tiles, 1)) != cudaSuccess)
    return NNP_ERR_CUDA;
  cudaMemset(tw->done, 0, sizeof(int) * (size_t)std::max(ws->max_tiles, 1));
  if (cudaMalloc(&tw->cscr, sizeof(uint32_t) * (size_t)TC_CSCR_WORDS * tw->num_sms) != cudaSuccess) return NNP_ERR_CUDA;
  return NNP_OK;
}

void tc_workspace_destroy(nnp_workspace* ws) {
  TcWorkspace* tw = static_cast<TcWorkspace*>(ws->tc_ws);
  if (!tw) return;
  for (int mem = 0; mem < MAX_MEMBERS; ++mem)
    for (int s = 0; s < MAX_S; ++s) {
      if (tw->w1img[mem][s]) cudaFree(tw->w1img[mem][s]);
      if (tw->w1timg[mem][s]) cudaFree(tw->w1timg[mem][s]);
    }
  if (tw->key) cudaFree(tw->key);
  if (tw->d_pall) cudaFree(tw->d_pall);
  if (tw->done) cudaFree(tw->done);
  if (tw->cscr) cudaFree(tw->cscr);
  cudaGetLastError();
  delete tw;
  ws->tc_ws = nullptr;
}

int tc_read_timeline(long long* h64) {
#ifdef NNP_TC_TIMELINE
  return cudaMemcpyFromSymbol(h64, g_tc_timeline, sizeof(long long) * 64) == cudaSuccess ? NNP_OK : NNP_ERR_CUDA;
#else
  (void)h64;
  return NNP_ERR_UNSUPPORTED;   // built without -DNNP_TC_TIMELINE
#endif
}

// Ensemble hand-over guard.  The members of a tile hand over between the CO-RESIDENT CTAs of one persistent launch: a
// CTA spins on done[tile] until the CTA holding the previous member releases it.  Two such launches running at the same
// time on different streams could each hold SMs the other's awaited CTA needs -- a deadlock.  The library therefore
// orders ensemble MLP launches across ALL workspaces of the process: every launch waits (cudaStreamWaitEvent) for the
// previous ensemble launch, whatever stream that was on, and records the event the next one waits for.  (Skipped while
// the stream is being captured into a CUDA graph: an event recorded outside the capture cannot be waited on inside it --
// replaying ensemble graphs concurrently on several streams stays the caller's responsibility.)
namespace {
std::mutex g_ens_mutex;
cudaEvent_t g_ens_event = nullptr;
bool g_ens_recorded = false;
}  // namespace

static void ensemble_guard_before(cudaStream_t st) {
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) { cudaGetLastError(); return; }
  std::lock_guard<std::mutex> lk(g_ens_mutex);
  if (g_ens_recorded) cudaStreamWaitEvent(st, g_ens_event, 0);
}
static void ensemble_guard_after(cudaStream_t st) {
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) { cudaGetLastError(); return; }
  std::lock_guard<std::mutex> lk(g_ens_mutex);
  if (!g_ens_event && cudaEventCreateWithFlags(&g_ens_event, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); g_ens_event = nullptr; return; }
  if (cudaEventRecord(g_ens_event, st) == cudaSuccess) g_ens_recorded = true; else cudaGetLastError();
}

// k_tc_pack_w1 needs the groups of this evaluation (k_cell_sort / k_prep / k_small_front) and must be through before the MLP
// kernel starts.  Directly in front of the MLP kernel it sits on the critical path (step timeline: the AEV kernel ends, the
// pack kernel's wait returns 1.1 us later, it runs 1 us, and only then do the MLP CTAs come in: 2.6 us); the cell-list path
// therefore launches it right after k_cell_sort, where it is a 1 us link in front of k_neighbors instead and its L2
// prefetch has the whole neighbour + AEV stage to land.  Returns the number of launches (0: no tensor-core MLP this time).
int launch_tc_pack(nnp_workspace* ws) {
  const nnp_model* m = ws->model;
  TcModel* tm = static_cast<TcModel*>(m->tc);
  TcWorkspace* tw = static_cast<TcWorkspace*>(ws->tc_ws);
  if (!tm || !tw || ws->mlp_mode == NNP_MLP_FP32_SIMT) return 0;
  TcPackAll pall;
  for (int mem = 0; mem < MAX_MEMBERS; ++mem)
    for (int s = 0; s < MAX_S; ++s) { pall.m[mem].w1[s] = tw->w1img[mem][s]; pall.m[mem].w1t[s] = tw->w1timg[mem][s]; }
  const bool pdl = !ws->profiling;
  // the operand prefetch pays for one network per element at compact K (~2 MB: step 249.2 -> 247.5 us); with eight members
  // (16 MB) or dense K (first-layer images of 1 MB each) it costs more in front of k_neighbors than it saves: +6 / +4 us
  const bool prefetch = pdl && m->n_members == 1 && !ws->dense_k;
  launch_pdl(pdl, ws->stream, k_tc_pack_w1, dim3(32, m->aev.S, m->n_members), dim3(256), 0, tm->d_nets, ws->groups, pall,
             tm->d_tabs, prefetch ? m->Kfull : 0, tw->key, tw->done, ws->max_tiles);
  ws->pack_done = 1;
  return 1;
}

int launch_mlp_tc(nnp_workspace* ws, int64_t n_ml) {
  if (n_ml <= 0) { ws->pack_done = 0; return 0; }
  const nnp_model* m = ws->model;
  TcModel* tm = static_cast<TcModel*>(m->tc);
  TcWorkspace* tw = static_cast<TcWorkspace*>(ws->tc_ws);
  if (!tm || !tw) return launch_mlp_simt(ws, n_ml);
  ws->tile_done = tw->done; ws->tile_done_target = m->n_members;
  int nl = 0;
  if (!ws->pack_done) nl += launch_tc_pack(ws);
  ws->pack_done = 0;
  const bool ens = m->n_members > 1;
  if (ens) ensemble_guard_before(ws->stream);
  // (a wait on another stream's event in front of the launch: no programmatic overlap with the predecessor then)
  const bool pdl = !ws->profiling;
  // one persistent CTA per SM over the (member, tile) work items (all CTAs are co-resident: 1 CTA/SM by shared memory)
  const int grid = (int)std::min<int64_t>((int64_t)ws->max_tiles * m->n_members, tw->num_sms);
  const float escale = 1.0f / (float)m->n_members;   // E = mean over the ensemble members
  if (ws->mlp_mode == NNP_MLP_F16X1)
    launch_pdl(pdl, ws->stream, k_mlp_tc<1>, dim3(grid), dim3(TC_THREADS), tw->smem_bytes[1], tm->d_nets, tm->d_tabs,
               tw->d_pall, ws->groups, ws->tiles, ws->aev, ws->daev, ws->e_atom, tw->key, tw->done, m->n_members, escale, tw->cscr);
  else
    launch_pdl(pdl, ws->stream, k_mlp_tc<3>, dim3(grid), dim3(TC_THREADS), tw->smem_bytes[0], tm->d_nets, tm->d_tabs,
               tw->d_pall, ws->groups, ws->tiles, ws->aev, ws->daev, ws->e_atom, tw->key, tw->done, m->n_members, escale, tw->cscr);
  if (ens) ensemble_guard_after(ws->stream);
  return nl + 1;
}

}  // namespace nnp

TL_EXPORT(nnp_debug_step_timeline_mlp)
