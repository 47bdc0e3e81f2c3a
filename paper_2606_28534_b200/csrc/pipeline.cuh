// Tile staging for the two particle passes: one tile (kTile particles: x, v, pid, species -- the cell index is
// cell_of(x) by construction and is not fetched --, its event bits and its window of E) is brought into shared memory by 1D bulk-async copies (TMA, SASS UBLKCP) that complete on an
// mbarrier, two stages deep, so that the next tile's 41 B x kTile are in flight while the current tile is computed.
// bytes in flight per SM are decoupled from registers and occupancy.
#pragma once
#include "common.cuh"

namespace bit1 {

struct __align__(128) Stage {
  double x[kTile], vx[kTile], vy[kTile], vz[kTile];
  unsigned pid[kTile];
  unsigned char sp[kTile];
  unsigned evt[kTile / 32];
  double E[kWCap + 4];  // E[e0 .. ], e0 = clo & ~1 (16-byte aligned source)
  int tb[kWCap];                  // pass B: the tile's row of tile_base
  unsigned pre[kWCap * kWarps];   // pass B: the tile's row of tile_pre
  int2 d;               // (first, last) old cell of the staged tile; plain store by the issuing thread
};

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long* b, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* b, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* b, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}\n" ::"r"(smem_u32(b)),
      "r"(parity)
      : "memory");
}
// global -> shared bulk copy; dst, src and bytes are multiples of 16
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* b) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(b))
               : "memory");
}
// orders this thread's generic-proxy accesses to shared memory before later async-proxy (TMA) writes
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// Split CTA barrier (named barriers 1 and 2): every warp but one announces that it is done with a tile and goes on; the
// one warp that owns the tile's hand-over waits for all of them.  Shared-memory accesses made before bar.arrive are
// visible after the matching bar.sync.
__device__ __forceinline__ void named_bar_arrive(int id, int nthreads) {
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// window of E that a tile with old cells [clo, chi] gathers from: E[clo .. chi+1]
__device__ __forceinline__ bool e_window(int clo, int chi, int& e0, int& ne) {
  e0 = clo & ~1;
  ne = (chi + 2 - e0 + 1) & ~1;
  return ne <= kWCap + 4;
}

// The sort window of a tile whose old cells are [clo, chi]: cells [wlo, wlo + W) with W <= kWCap.  The radius is the
// step's R (DevState::R_cur), cut down symmetrically for tiles so sparse that the window would not fit.  Pass A,
// k_mid and pass B all derive a tile's window through this one function.
struct TileWin {
  int clo, chi, wlo, W;
};
__device__ __forceinline__ TileWin make_window(int clo, int chi, int R) {
  TileWin t;
  const int span = chi - clo + 1;
  if (span + 2 * R > kWCap) R = span < kWCap ? (kWCap - span) >> 1 : 0;
  t.clo = clo; t.chi = chi; t.wlo = clo - R;
  const int w = span + 2 * R;
  t.W = w < kWCap ? w : kWCap;
  return t;
}

// One elected thread: arm the stage's barrier and issue the copies of tile `tile` (always whole tiles: the
// arrays are padded to a multiple of kTile, the tail of the last tile is never used).
__device__ __forceinline__ void issue_tile(const Params& P, const Particles& cur, Stage* st, unsigned long long* bar,
                                           int tile, int2 d, int R, bool with_evt, bool with_E, bool with_rank) {
  const size_t base = (size_t)tile * kTile;
  int e0 = 0, ne = 0;
  const bool stage_E = with_E && e_window(d.x, d.y, e0, ne);
  unsigned bytes = 4u * kTile * 8u + kTile * 4u + kTile;
  if (with_evt) bytes += kTile / 8;
  if (stage_E) bytes += (unsigned)ne * 8u;
  // window of the tile, rounded up to whole 16-byte units (the rows are padded, see tile_row_offset)
  const int w = (make_window(d.x, d.y, R).W + 3) & ~3;
  const size_t row = tile_row_offset(d.x, tile, R);
  if (with_rank) bytes += (unsigned)w * 4u * (1u + (unsigned)kWarps);
  st->d = d;
  mbar_expect_tx(bar, bytes);
  bulk_g2s(st->x, cur.x + base, kTile * 8, bar);
  bulk_g2s(st->vx, cur.vx + base, kTile * 8, bar);
  bulk_g2s(st->vy, cur.vy + base, kTile * 8, bar);
  bulk_g2s(st->vz, cur.vz + base, kTile * 8, bar);
  bulk_g2s(st->pid, cur.pid + base, kTile * 4, bar);
  bulk_g2s(st->sp, cur.sp + base, kTile, bar);
  if (with_evt) bulk_g2s(st->evt, P.evt + base / 32, kTile / 8, bar);
  if (stage_E) bulk_g2s(st->E, P.E + e0, (unsigned)ne * 8u, bar);
  if (with_rank) {
    bulk_g2s(st->tb, P.tile_base + row, (unsigned)w * 4u, bar);
    bulk_g2s(st->pre, P.tile_pre + row * kWarps, (unsigned)w * 4u * (unsigned)kWarps, bar);
  }
}

}  // namespace bit1
