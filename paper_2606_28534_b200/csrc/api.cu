// C ABI of libbit1 (include/bit1.h): argument checking, workspace layout, stream-ordered launches.
// Every step of the hot path runs in the kernels of step_kernels.cu; nothing here computes on the host
// beyond the derived constants of DESIGN.md "Derived constants".
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <atomic>
#include <new>
#include <vector>

#include <nvtx3/nvToolsExt.h>   // header-only; ranges show up in Nsight Systems timelines (PAPER.md:105-113 used the same)

#include "../../include/bit1.h"
#include "aux_kernels.h"
#include "step_kernels.h"

using namespace bit1;

namespace {

constexpr double kECharge = 1.602176634e-19;   // C, CODATA 2018
constexpr double kEps0 = 8.8541878128e-12;     // F/m
constexpr double kTwoM40 = 9.094947017729282379150390625e-13;
constexpr int kMaxSig = 16384;
constexpr int kMaxNorm = 1 << 20;
constexpr int kDefaultRmax = 16;
constexpr size_t kAlign = 256;
// 2: + averaging sums (NEXT-1); 3: + recycling counter (NEXT-2); 4: live prefix only, no cell array, no cell_start
constexpr uint32_t kCkptVersion = 4;

// settings of bit1_options that shape the workspace
struct Shape {
  size_t cap;        // particle capacity
  int staging;       // device snapshot area for overlapped checkpoints
  int r_max;         // upper bound of the adaptive sort-window radius
  size_t ovf_cap;    // side-list capacity
};
inline bool shape_of(const bit1_options* o, Shape* sh) {
  if (!o || o->capacity == 0 || o->capacity >= (1ull << 31)) return false;
  sh->cap = (size_t)o->capacity;
  sh->staging = o->checkpoint_staging ? 1 : 0;
  sh->r_max = o->window_radius_max == 0 ? kDefaultRmax : o->window_radius_max;
  if (sh->r_max < 1 || sh->r_max > kMaxR) return false;
  if (o->window_radius_fixed < 0 || o->window_radius_fixed > kMaxR + 1) return false;
  if (o->window_radius_fixed > 0 && o->window_radius_fixed - 1 > sh->r_max) sh->r_max = o->window_radius_fixed - 1;
  if (sh->r_max < 1) sh->r_max = 1;
  size_t oc = o->side_list_capacity;
  if (oc == 0) { oc = sh->cap / 16; if (oc < 65536) oc = 65536; }
  if (oc < 16 || oc >= (1ull << 31)) return false;
  sh->ovf_cap = oc;
  return true;
}

inline size_t align_up(size_t v) { return (v + kAlign - 1) & ~(kAlign - 1); }

struct PartLayout {
  size_t x, vx, vy, vz, cell, pid, sp, desc, bytes;
};
// every array holds a whole number of tiles: the bulk-async loads always fetch whole tiles
PartLayout part_layout(size_t cap_in) {
  PartLayout l;
  const size_t tiles = (cap_in + kTile - 1) / kTile;
  const size_t cap = tiles * kTile;
  size_t o = 0;
  l.x = o; o += align_up(cap * 8);
  l.vx = o; o += align_up(cap * 8);
  l.vy = o; o += align_up(cap * 8);
  l.vz = o; o += align_up(cap * 8);
  l.cell = o; o += align_up(cap * 4);
  l.pid = o; o += align_up(cap * 4);
  l.sp = o; o += align_up(cap);
  l.desc = o; o += align_up((tiles + 1) * 8);
  l.bytes = o;
  return l;
}
Particles part_at(void* base, const PartLayout& l) {
  char* b = static_cast<char*>(base);
  Particles p;
  p.x = reinterpret_cast<double*>(b + l.x);
  p.vx = reinterpret_cast<double*>(b + l.vx);
  p.vy = reinterpret_cast<double*>(b + l.vy);
  p.vz = reinterpret_cast<double*>(b + l.vz);
  p.cell = reinterpret_cast<int*>(b + l.cell);
  p.pid = reinterpret_cast<unsigned*>(b + l.pid);
  p.sp = reinterpret_cast<unsigned char*>(b + l.sp);
  p.desc = reinterpret_cast<int2*>(b + l.desc);
  return p;
}

// running + latched sums of the time-averaged diagnostics, one contiguous block:
// acc_dens[ns*ng] | avg_dens[ns*ng] (int64) | acc_phi[nc+1] | avg_phi[nc+1] (fp64)
size_t avg_bytes(int nc, int ng, int ns) { return 2 * ((size_t)ns * ng + (size_t)(nc + 1)) * 8; }

// Checkpoint blob: header | DevState | averaging sums | x | vx | vy | vz | pid |
// species, each array holding the n live particles only (256-byte aligned).  The cell index and the counts per cell
// are functions of x and are rebuilt at restart.
struct CkptLayout {
  size_t header, state, avg, x, vx, vy, vz, pid, sp, bytes;
};
CkptLayout ckpt_layout(int nc, int ng, int ns, size_t n) {
  CkptLayout c;
  c.header = 0;
  c.state = 256;
  c.avg = c.state + align_up(sizeof(DevState));
  size_t o = c.avg + align_up(avg_bytes(nc, ng, ns));
  c.x = o; o += align_up(n * 8);
  c.vx = o; o += align_up(n * 8);
  c.vy = o; o += align_up(n * 8);
  c.vz = o; o += align_up(n * 8);
  c.pid = o; o += align_up(n * 4);
  c.sp = o; o += align_up(n);
  c.bytes = o;
  return c;
}

// Streamed snapshot (bit1_stream_publish): per species the counts per cell (int32[nc]) and the x, vx, vy, vz (fp64)
// and id (uint32) records in cell order, every array 256-byte aligned; worst case over how n splits among species
size_t stream_payload_bytes(int nc, int ns, size_t n) {
  return (size_t)ns * (align_up((size_t)nc * 4) + 5 * kAlign) + 4 * align_up(n * 8) + align_up(n * 4) +
         (size_t)ns * 5 * kAlign;
}

struct Layout {
  size_t st, tables, dens, dens_old, rho, rho_s, rho_t, avg, phi, E, cell_count, cell_start, cell_start_old, scan_part, coop_scratch, cell_base, ovf_before, ovf_lb, ovf_ub, radix_hist, tile_hist, tile_base, tile_pre, evt,
      ovf_key, ovf_idx, ovf_dst, tmp_key, tmp_idx, tmp2_key, tmp2_idx, ovf_rec, part[2], scratch, small, exp, mom, total;
  unsigned ovf_cap;
  int max_tiles, ng;
  size_t scratch_bytes;
};
Layout make_layout(int nc, int bc, int ns, const Shape& sh) {
  Layout l;
  const size_t cap = sh.cap;
  l.ng = bc ? nc + 1 : nc;
  l.max_tiles = (int)((cap + kTile - 1) / kTile);
  l.ovf_cap = (unsigned)sh.ovf_cap;
  const size_t oc = l.ovf_cap;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o += align_up(bytes); return at; };
  l.st = take(sizeof(DevState));
  l.tables = take(((size_t)3 * kMaxSig + kMaxNorm + 1) * 8);
  l.dens = take((size_t)ns * l.ng * 8);
  l.dens_old = take((size_t)ns * l.ng * 8);
  l.rho = take((size_t)l.ng * 8);
  l.rho_s = take((size_t)l.ng * 8);
  l.rho_t = take((size_t)l.ng * 8);
  l.avg = take(avg_bytes(nc, l.ng, ns));
  l.phi = take((size_t)(nc + 1) * 8);
  l.E = take((size_t)(nc + 4) * 8);  // the E window of a tile is copied in 16-byte units
  l.cell_count = take((size_t)nc * 4);
  l.cell_start = take((size_t)(nc + 1) * 4);
  l.cell_start_old = take((size_t)(nc + 1) * 4);
  l.scan_part = take(1024 * 4);
  l.coop_scratch = take(4 * 1024 * 16);
  l.cell_base = take((size_t)nc * 4);
  l.ovf_before = take((size_t)nc * 4);
  l.ovf_lb = take((size_t)nc * 4);
  l.ovf_ub = take((size_t)nc * 4);
  l.radix_hist = take((size_t)256 * 256 * 4);
  const size_t rw = tile_row_words(nc, l.max_tiles, sh.r_max);
  l.tile_hist = take(rw * 4);
  l.tile_base = take(rw * 4);
  l.tile_pre = take(rw * 4 * kWarps);
  l.evt = take((size_t)(l.max_tiles + 1) * (kTile / 8));
  l.ovf_key = take(oc * 8);
  l.tmp_key = take(oc * 8);
  l.tmp2_key = take(oc * 8);
  l.ovf_idx = take(oc * 4);
  l.ovf_dst = take(oc * 4);
  l.tmp_idx = take(oc * 4);
  l.tmp2_idx = take(oc * 4);
  l.ovf_rec = take(oc * sizeof(OvfRec));
  const PartLayout pl = part_layout(cap);
  l.part[0] = take(pl.bytes);
  l.part[1] = take(pl.bytes);
  // one scratch area for the calls that never overlap one another: load-time sort, general-path step, export, and
  // the device snapshot of an overlapped checkpoint (a general-path step first waits for a pending checkpoint)
  l.scratch_bytes = general_scratch_bytes((unsigned)cap);
  if (sh.staging) {
    size_t cb = ckpt_layout(nc, l.ng, ns, cap).bytes;
    const size_t sb = stream_payload_bytes(nc, ns, cap);   // bit1_stream_publish stages its records there too
    if (sb > cb) cb = sb;
    if (cb > l.scratch_bytes) l.scratch_bytes = cb;
  }
  l.scratch = take(l.scratch_bytes);
  l.exp = take(export_scratch_bytes(nc, (unsigned)cap));
  l.small = take(ckpt_layout(nc, l.ng, ns, 0).bytes);   // DevState + averaging sums of a checkpoint without staging
  l.mom = take(moments_scratch_bytes());
  l.total = o;
  return l;
}

struct CkptHeader {
  char magic[8];
  uint32_t version;
  int32_t nc, ns, bc;
  uint64_t capacity, cfg_hash, bytes, n;
};

uint64_t fnv1a(uint64_t h, const void* data, size_t n) {
  const unsigned char* p = static_cast<const unsigned char*>(data);
  for (size_t i = 0; i < n; ++i) { h ^= p[i]; h *= 1099511628211ull; }
  return h;
}

}  // namespace

namespace {
struct NvtxRange {   // RAII range around an entry point
  explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
  ~NvtxRange() { nvtxRangePop(); }
};
}  // namespace

struct bit1_ctx {
  Params P;
  Layout lay;
  Shape shape;
  Particles buf[2];
  int cur;
  char* ws;
  cudaStream_t cs, ss;
  cudaEvent_t ev_snap, ev_done, ev_load0, ev_load1[3];
  bool ckpt_pending, staging, loaded;
  bool ckpt_reads_live;   // a checkpoint without staging is still copying out of the live half of the store
  uint64_t launches, cfg_hash, cfg_hash_base;
  double m[BIT1_MAX_SPECIES], weight[BIT1_MAX_SPECIES];
  double dt;
  bool profiling;
  // two timesteps captured as one CUDA graph per starting parity of the ping-pong buffers (small workloads are bound by
  // launch overhead: 8-10 launches, two of them cooperative, replayed with one call)
  cudaGraphExec_t graph[2];
  bool use_graph;
  std::vector<cudaEvent_t> prof_ev;  // 5 per timed step
  size_t prof_steps;
  // Steps are enqueued without looking at the device.  step_target is the value the device's step counter has
  // when everything enqueued has really run; a step whose side list did not fit stalls on the device (it and the
  // steps behind it return at once) and settle() takes it through the general path at the next call that waits.
  uint64_t step_target;
  uint64_t last_general_step;   // step index the general path last took
  unsigned burst;               // steps to take by the general path outright after the next stall
  uint64_t general_steps_host;
  // streaming checkpoints (bit1_stream_*): ring of caller-owned pinned slots, states shared with the consumer thread
  char* ring;
  size_t slot_bytes;
  int nslots;
  uint64_t next_seq;
  std::atomic<int> slot_state[BIT1_STREAM_MAX_SLOTS];        // kSlotFree / Filling / Ready / Held
  std::atomic<uint64_t> slot_seq[BIT1_STREAM_MAX_SLOTS];
  struct StreamDone { bit1_ctx* c; int slot; uint64_t seq; } done_arg[BIT1_STREAM_MAX_SLOTS];
};
enum { kSlotFree = 0, kSlotFilling = 1, kSlotReady = 2, kSlotHeld = 3 };
constexpr size_t kMaxProfSteps = 4096;

#define CUDA_OK(call)                              \
  do {                                             \
    cudaError_t e_ = (call);                       \
    if (e_ != cudaSuccess) return BIT1_ERR_CUDA;   \
  } while (0)
#define BIT1_OK_OR_RETURN(call)                    \
  do {                                             \
    bit1_status s_ = (call);                       \
    if (s_ != BIT1_OK) return s_;                  \
  } while (0)

// configuration hash: recomputed from the base hash and the NEXT-2 settings, so the order of the calls is irrelevant
static void rehash(bit1_ctx* c) {
  uint64_t h = c->cfg_hash_base;
  for (int s = 0; s < c->P.ns; ++s) {
    h = fnv1a(h, &c->P.sp[s].recycle_to, 4);
    h = fnv1a(h, &c->P.sp[s].recycle_vth, 8);
  }
  h = fnv1a(h, &c->P.target_species, 4);
  c->cfg_hash = h;
}

static int bits_for(unsigned long long v) {   // bits needed to write values 0 .. v
  int b = 1;
  while (b < 63 && (v >> b) != 0ull) ++b;
  return b;
}

extern "C" {

const char* bit1_error_string(bit1_status s) {
  switch (s) {
    case BIT1_OK: return "ok";
    case BIT1_ERR_INVALID_ARG: return "invalid argument";
    case BIT1_ERR_RANGE: return "fixed-point charge out of range [1, 2^31)";
    case BIT1_ERR_CAPACITY: return "capacity or workspace too small";
    case BIT1_ERR_STATE: return "call out of order";
    case BIT1_ERR_CUDA: return "CUDA runtime error or no device";
    case BIT1_ERR_CHECKPOINT: return "checkpoint blob does not match this context";
    case BIT1_ERR_DEVICE_FLAG: return "sticky device flag set";
    case BIT1_ERR_STATIC_LIMIT:
      return "grid has more cells than the built-in scratch of bit1_field_solve_static holds (BIT1_FIELD_STATIC_MAX_CELLS = 1048576)";
  }
  return "unknown";
}

size_t bit1_workspace_size(const bit1_grid* g, int ns, const bit1_options* o) {
  Shape sh;
  if (!g || g->nc < 2 || g->nc >= (1 << 28) || ns < 1 || ns > BIT1_MAX_SPECIES || !shape_of(o, &sh)) return 0;
  return make_layout(g->nc, g->bc, ns, sh).total;
}

bit1_status bit1_create(const bit1_grid* g, const bit1_species* sp, int ns, double dt, const bit1_options* o,
                        bit1_ctx** out) {
  if (!g || !sp || !o || !out) return BIT1_ERR_INVALID_ARG;
  if (g->nc < 2 || g->nc >= (1 << 28) || (g->bc != 0 && g->bc != 1) || !(g->dx > 0.0) || !(g->area > 0.0) ||
      !(dt > 0.0) || ns < 1 || ns > BIT1_MAX_SPECIES)
    return BIT1_ERR_INVALID_ARG;
  Shape sh;
  if (!shape_of(o, &sh)) return BIT1_ERR_INVALID_ARG;
  if (o->launch_mode != 0 && o->launch_mode != 1) return BIT1_ERR_INVALID_ARG;
  if (o->n_sig < 0 || o->n_sig > kMaxSig || o->n_norm < 1 || o->n_norm > kMaxNorm || !o->inv_norm)
    return BIT1_ERR_INVALID_ARG;
  if (!o->workspace || (reinterpret_cast<uintptr_t>(o->workspace) & (kAlign - 1))) return BIT1_ERR_INVALID_ARG;
  int sp_ep = -1, sp_ip = -1;
  bool any_coll = false, any_ion = false, any_src = false;
  for (int s = 0; s < ns; ++s) {
    if (!(sp[s].m > 0.0) || !(sp[s].weight > 0.0)) return BIT1_ERR_INVALID_ARG;
    if (sp[s].src_mode < 0 || sp[s].src_mode > 2) return BIT1_ERR_INVALID_ARG;
    if (sp[s].src_mode == BIT1_SRC_PAIR && (sp[s].src_partner < 0 || sp[s].src_partner >= ns))
      return BIT1_ERR_INVALID_ARG;
    if (sp[s].src_mode != BIT1_SRC_NONE) any_src = true;
    if ((sp[s].flags & BIT1_ELECTRON_PRODUCT) && sp_ep < 0) sp_ep = s;
    if ((sp[s].flags & BIT1_ION_PRODUCT) && sp_ip < 0) sp_ip = s;
    if (sp[s].flags & (BIT1_ELASTIC | BIT1_IONISE | BIT1_CX)) any_coll = true;
    if (sp[s].flags & BIT1_IONISE) any_ion = true;
  }
  if (any_coll && (o->n_sig < 2 || !o->sig_el || !o->sig_ion || !o->sig_cx || !(o->dE_eV > 0.0) || !(o->m_n > 0.0)))
    return BIT1_ERR_INVALID_ARG;
  if (any_ion && (sp_ep < 0 || sp_ip < 0 || sp[sp_ep].weight != sp[sp_ip].weight)) return BIT1_ERR_INVALID_ARG;
  // a re-injection source only acts at absorbing walls and must put particles inside the domain
  if (any_src && g->bc == 1 &&
      !(o->src_lo >= 0.0 && o->src_lo < o->src_hi && o->src_hi <= (double)g->nc * g->dx))
    return BIT1_ERR_INVALID_ARG;

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return BIT1_ERR_CUDA;

  const Layout lay = make_layout(g->nc, g->bc, ns, sh);
  if (o->workspace_bytes < lay.total) return BIT1_ERR_CAPACITY;

  bit1_ctx* c = new (std::nothrow) bit1_ctx();
  if (!c) return BIT1_ERR_INVALID_ARG;
  memset(&c->P, 0, sizeof(Params));
  c->lay = lay;
  c->shape = sh;
  c->ws = static_cast<char*>(o->workspace);
  c->cs = static_cast<cudaStream_t>(o->compute_stream);
  c->ss = o->side_stream ? static_cast<cudaStream_t>(o->side_stream) : c->cs;
  c->staging = sh.staging != 0;
  c->cur = 0; c->loaded = false; c->ckpt_pending = false; c->ckpt_reads_live = false; c->launches = 0; c->dt = dt;
  c->profiling = false; c->prof_steps = 0;
  c->graph[0] = c->graph[1] = nullptr;
  c->use_graph = o->launch_mode == 0;
  c->step_target = 0; c->last_general_step = ~0ull; c->burst = 0; c->general_steps_host = 0;
  c->ring = nullptr; c->slot_bytes = 0; c->nslots = 0; c->next_seq = 1;
  for (int k = 0; k < BIT1_STREAM_MAX_SLOTS; ++k) { c->slot_state[k].store(kSlotFree); c->slot_seq[k].store(0); }

  Params& P = c->P;
  P.nc = g->nc; P.bc = g->bc; P.ng = lay.ng; P.ns = ns;
  P.R_max = sh.r_max;
  P.R_fixed = o->window_radius_fixed > 0 ? o->window_radius_fixed - 1 : -1;
  // side-list key: cell | class (2 bits) | order (array index * 4 + birth kind)
  P.ord_bits = bits_for((unsigned long long)sh.cap * 4ull + 3ull);
  P.cell_shift = P.ord_bits + 2;
  P.key_bits = P.cell_shift + bits_for((unsigned long long)(g->nc - 1));
  P.n_sig = o->n_sig; P.n_norm = o->n_norm; P.sp_ep = sp_ep; P.sp_ip = sp_ip;
  P.seed_lo = (unsigned)o->seed; P.seed_hi = (unsigned)(o->seed >> 32);
  P.capacity = (unsigned)o->capacity; P.ovf_cap = lay.ovf_cap;
  P.max_tiles = lay.max_tiles;
  // derived constants, one documented expression each
  P.inv_dx = 1.0 / g->dx;
  P.L = (double)g->nc * g->dx;
  P.dt = dt; P.dx = g->dx; P.area = g->area;
  P.src_lo = o->src_lo; P.src_span = o->src_hi - o->src_lo;
  P.n0 = o->n0; P.vth_n = o->vth_n; P.E_ion = o->E_ion; P.dE_eV = o->dE_eV;
  P.Kphi = (kTwoM40 * g->dx) / ((g->area * kEps0) * (double)g->nc);
  P.KE = kTwoM40 / (((2.0 * (double)g->nc) * g->area) * kEps0);
  if (!g->bc) { P.Kphi = P.Kphi / (double)g->nc; P.KE = P.KE / (double)g->nc; }
  P.field_J_factor = ((0.5 * kEps0) * g->area) * g->dx;
  P.dep_u32 = 1;
  const double B[3] = {g->Bx, g->By, g->Bz};
  for (int s = 0; s < ns; ++s) {
    SpeciesP& q = P.sp[s];
    const double h = 0.5 * ((sp[s].q / sp[s].m) * dt);
    q.h = h;
    q.tx = h * B[0]; q.ty = h * B[1]; q.tz = h * B[2];
    const double tt = (q.tx * q.tx + q.ty * q.ty) + q.tz * q.tz;
    q.sx = (2.0 * q.tx) / (1.0 + tt);
    q.sy = (2.0 * q.ty) / (1.0 + tt);
    q.sz = (2.0 * q.tz) / (1.0 + tt);
    q.src_vth = sp[s].src_vth; q.pnull = sp[s].pnull; q.numax = sp[s].numax;
    // integer form of the candidate test: the uniform is u = (w + 0.5) * 2^-52 with a 52-bit integer w (exact),
    // so u < pnull  <=>  w + 0.5 < y = pnull * 2^52 (exact scaling)  <=>  w < floor(y) + (frac(y) > 0.5)
    q.pthr = 0;
    if ((sp[s].flags & (BIT1_ELASTIC | BIT1_IONISE | BIT1_CX)) && sp[s].pnull > 0.0) {
      const double y = (sp[s].pnull < 1.0 ? sp[s].pnull : 1.0) * 4503599627370496.0;
      const double fl = floor(y);
      q.pthr = (unsigned long long)fl + ((y - fl) > 0.5 ? 1ull : 0ull);
    }
    q.kin_eV = (0.5 * sp[s].m) / kECharge;
    q.two_e_over_m = (2.0 * kECharge) / sp[s].m;
    q.el_loss = o->m_n > 0.0 ? (2.0 * sp[s].m) / o->m_n : 0.0;
    q.Q = llrint((kECharge * sp[s].weight) * 1099511627776.0);
    q.sign = sp[s].q > 0.0 ? 1 : (sp[s].q < 0.0 ? -1 : 0);
    q.flags = sp[s].flags; q.src_mode = sp[s].src_mode; q.src_partner = sp[s].src_partner;
    q.recycle_to = -1; q.recycle_vth = 0.0;
    if (q.Q < 1 || q.Q >= (1ll << 31)) { delete c; return BIT1_ERR_RANGE; }
    if ((unsigned long long)q.Q * (unsigned long long)kTile >= (1ull << 32) || q.Q >= (1ll << 21)) P.dep_u32 = 0;
    c->m[s] = sp[s].m; c->weight[s] = sp[s].weight;
  }
  char* ws = c->ws;
  P.st = reinterpret_cast<DevState*>(ws + lay.st);
  double* tab = reinterpret_cast<double*>(ws + lay.tables);
  P.sig_el = tab; P.sig_ion = tab + kMaxSig; P.sig_cx = tab + 2 * kMaxSig; P.inv_norm = tab + 3 * kMaxSig;
  P.dens = reinterpret_cast<long long*>(ws + lay.dens);
  P.dens_old = reinterpret_cast<long long*>(ws + lay.dens_old);
  P.target_species = -1; P.kn = 0.0;
  P.rho = reinterpret_cast<long long*>(ws + lay.rho);
  P.rho_s = reinterpret_cast<long long*>(ws + lay.rho_s);
  P.rho_t = reinterpret_cast<long long*>(ws + lay.rho_t);
  P.acc_dens = reinterpret_cast<long long*>(ws + lay.avg);
  P.avg_dens = P.acc_dens + (size_t)ns * lay.ng;
  P.acc_phi = reinterpret_cast<double*>(P.avg_dens + (size_t)ns * lay.ng);
  P.avg_phi = P.acc_phi + (g->nc + 1);
  P.phi = reinterpret_cast<double*>(ws + lay.phi);
  P.E = reinterpret_cast<double*>(ws + lay.E);
  P.cell_count = reinterpret_cast<int*>(ws + lay.cell_count);
  P.cell_start = reinterpret_cast<int*>(ws + lay.cell_start);
  P.cell_start_old = reinterpret_cast<int*>(ws + lay.cell_start_old);
  P.scan_part = reinterpret_cast<int*>(ws + lay.scan_part);
  P.coop_scratch = ws + lay.coop_scratch;
  P.cell_base = reinterpret_cast<int*>(ws + lay.cell_base);
  P.ovf_before = reinterpret_cast<int*>(ws + lay.ovf_before);
  P.ovf_lb = reinterpret_cast<int*>(ws + lay.ovf_lb);
  P.ovf_ub = reinterpret_cast<int*>(ws + lay.ovf_ub);
  P.radix_hist = reinterpret_cast<unsigned*>(ws + lay.radix_hist);
  P.tile_base = reinterpret_cast<int*>(ws + lay.tile_base);
  P.evt = reinterpret_cast<unsigned*>(ws + lay.evt);
  P.tile_hist = reinterpret_cast<unsigned*>(ws + lay.tile_hist);
  P.tile_pre = reinterpret_cast<unsigned*>(ws + lay.tile_pre);
  P.ovf_key = reinterpret_cast<unsigned long long*>(ws + lay.ovf_key);
  P.tmp_key = reinterpret_cast<unsigned long long*>(ws + lay.tmp_key);
  P.tmp2_key = reinterpret_cast<unsigned long long*>(ws + lay.tmp2_key);
  P.ovf_idx = reinterpret_cast<unsigned*>(ws + lay.ovf_idx);
  P.ovf_dst = reinterpret_cast<int*>(ws + lay.ovf_dst);
  P.tmp_idx = reinterpret_cast<unsigned*>(ws + lay.tmp_idx);
  P.tmp2_idx = reinterpret_cast<unsigned*>(ws + lay.tmp2_idx);
  P.ovf_rec = reinterpret_cast<OvfRec*>(ws + lay.ovf_rec);
  const PartLayout pl = part_layout((size_t)o->capacity);
  c->buf[0] = part_at(ws + lay.part[0], pl);
  c->buf[1] = part_at(ws + lay.part[1], pl);

  // configuration hash for checkpoint validation
  uint64_t h = 1469598103934665603ull;
  h = fnv1a(h, g, sizeof(*g));
  h = fnv1a(h, &dt, sizeof(dt));
  for (int s = 0; s < ns; ++s) {
    h = fnv1a(h, &sp[s].q, 8); h = fnv1a(h, &sp[s].m, 8); h = fnv1a(h, &sp[s].weight, 8);
    h = fnv1a(h, &sp[s].flags, 4); h = fnv1a(h, &sp[s].src_mode, 4); h = fnv1a(h, &sp[s].src_partner, 4);
    h = fnv1a(h, &sp[s].src_vth, 8); h = fnv1a(h, &sp[s].pnull, 8); h = fnv1a(h, &sp[s].numax, 8);
  }
  h = fnv1a(h, &o->seed, 8); h = fnv1a(h, &o->capacity, 8);
  h = fnv1a(h, &o->src_lo, 8); h = fnv1a(h, &o->src_hi, 8); h = fnv1a(h, &o->n0, 8);
  h = fnv1a(h, &o->vth_n, 8); h = fnv1a(h, &o->E_ion, 8); h = fnv1a(h, &o->m_n, 8); h = fnv1a(h, &o->dE_eV, 8);
  if (o->n_sig > 0 && o->sig_el) {
    h = fnv1a(h, o->sig_el, (size_t)o->n_sig * 8);
    h = fnv1a(h, o->sig_ion, (size_t)o->n_sig * 8);
    h = fnv1a(h, o->sig_cx, (size_t)o->n_sig * 8);
  }
  h = fnv1a(h, o->inv_norm, (size_t)(o->n_norm + 1) * 8);
  c->cfg_hash_base = h;
  rehash(c);   // the NEXT-2 settings (bit1_set_recycling, bit1_set_neutral_target) are hashed on top of the base

  bool ok = true;
  ok = ok && cudaMemsetAsync(ws + lay.st, 0, lay.part[0] - lay.st, c->cs) == cudaSuccess;  // state, grids, lists
  if (o->n_sig > 0 && o->sig_el) {
    ok = ok && cudaMemcpyAsync((void*)P.sig_el, o->sig_el, (size_t)o->n_sig * 8, cudaMemcpyHostToDevice, c->cs) == cudaSuccess;
    ok = ok && cudaMemcpyAsync((void*)P.sig_ion, o->sig_ion, (size_t)o->n_sig * 8, cudaMemcpyHostToDevice, c->cs) == cudaSuccess;
    ok = ok && cudaMemcpyAsync((void*)P.sig_cx, o->sig_cx, (size_t)o->n_sig * 8, cudaMemcpyHostToDevice, c->cs) == cudaSuccess;
  }
  ok = ok && cudaMemcpyAsync((void*)P.inv_norm, o->inv_norm, (size_t)(o->n_norm + 1) * 8, cudaMemcpyHostToDevice, c->cs) == cudaSuccess;
  ok = ok && cudaStreamSynchronize(c->cs) == cudaSuccess;
  ok = ok && configure_kernels() == cudaSuccess;
  ok = ok && cudaEventCreateWithFlags(&c->ev_snap, cudaEventDisableTiming) == cudaSuccess;
  ok = ok && cudaEventCreateWithFlags(&c->ev_done, cudaEventDisableTiming) == cudaSuccess;
  ok = ok && cudaEventCreateWithFlags(&c->ev_load0, cudaEventDisableTiming) == cudaSuccess;
  for (int k = 0; k < 3; ++k) ok = ok && cudaEventCreateWithFlags(&c->ev_load1[k], cudaEventDisableTiming) == cudaSuccess;
  if (!ok) { delete c; return BIT1_ERR_CUDA; }
  *out = c;
  return BIT1_OK;
}

// the captured launches hold the settings by value: any change to them drops the graphs
static void drop_graphs(bit1_ctx* c) {
  for (int k = 0; k < 2; ++k)
    if (c->graph[k]) { cudaGraphExecDestroy(c->graph[k]); c->graph[k] = nullptr; }
}

void bit1_destroy(bit1_ctx* c) {
  if (!c) return;
  cudaStreamSynchronize(c->cs);
  drop_graphs(c);
  if (c->ss != c->cs) cudaStreamSynchronize(c->ss);
  cudaEventDestroy(c->ev_snap);
  cudaEventDestroy(c->ev_done);
  cudaEventDestroy(c->ev_load0);
  for (int k = 0; k < 3; ++k) cudaEventDestroy(c->ev_load1[k]);
  for (cudaEvent_t e : c->prof_ev) cudaEventDestroy(e);
  delete c;
}

uint64_t bit1_launch_count(bit1_ctx* c) { return c ? c->launches : 0; }

int bit1_build_is_checked(void) {
#ifdef BIT1_CHECKED
  return 1;
#else
  return 0;
#endif
}

bit1_status bit1_check_selftest(bit1_ctx* c) {
  if (!c) return BIT1_ERR_INVALID_ARG;
#ifdef BIT1_CHECKED
  CUDA_OK(cudaStreamSynchronize(c->cs));
  DevState before, after;
  CUDA_OK(cudaMemcpy(&before, c->P.st, sizeof(DevState), cudaMemcpyDeviceToHost));
  launch_check_selftest(c->P, c->cs);
  CUDA_OK(cudaStreamSynchronize(c->cs));
  CUDA_OK(cudaMemcpy(&after, c->P.st, sizeof(DevState), cudaMemcpyDeviceToHost));
  const bool caught = after.check_count == before.check_count + 1 && (after.flags & kFlagCheck) &&
                      (before.check_count != 0 || (after.check_idx == 5 && after.check_limit == 3));
  CUDA_OK(cudaMemcpy(c->P.st, &before, sizeof(DevState), cudaMemcpyHostToDevice));   // clear the record again
  return caught ? BIT1_OK : BIT1_ERR_CUDA;
#else
  return BIT1_ERR_STATE;
#endif
}

bit1_status bit1_profile(bit1_ctx* c, int enable) {
  if (!c) return BIT1_ERR_INVALID_ARG;
  c->profiling = enable != 0;
  c->prof_steps = 0;
  return BIT1_OK;
}

static bit1_status read_state(bit1_ctx* c, DevState* h) {
  CUDA_OK(cudaMemcpyAsync(h, c->P.st, sizeof(DevState), cudaMemcpyDeviceToHost, c->cs));
  CUDA_OK(cudaStreamSynchronize(c->cs));
  return BIT1_OK;
}

// ---- enqueueing steps ---------------------------------------------------------------------------------------
// host-side view of "which half of the store, which cell_start, which dens is this step's input": flips every step
static void flip_parity(bit1_ctx* c) {
  { int* t = c->P.cell_start; c->P.cell_start = c->P.cell_start_old; c->P.cell_start_old = t; }
  { long long* t = c->P.dens; c->P.dens = c->P.dens_old; c->P.dens_old = t; }
  c->cur ^= 1;
}

// one timestep enqueued on the compute stream (also under stream capture)
static void enqueue_step(bit1_ctx* c, cudaEvent_t* ev) {
  // the arrangement the last step (or load / restart) produced is this step's input
  const int in = c->cur;
  flip_parity(c);
  c->launches += launch_step(c->P, c->buf[in], c->buf[in ^ 1], c->cs, ev);
}

// one timestep by the general path (general_kernels.cu)
static bit1_status enqueue_general_step(bit1_ctx* c, int count_side_effects) {
  if (c->ckpt_pending) {   // the scratch area may hold a checkpoint's device snapshot that is still being copied out
    CUDA_OK(cudaEventSynchronize(c->ev_done));
    c->ckpt_pending = false;
    c->ckpt_reads_live = false;
  }
  const int in = c->cur;
  flip_parity(c);
  c->launches += launch_general_step(c->P, c->buf[in], c->buf[in ^ 1], count_side_effects, c->ws + c->lay.scratch, c->cs);
  c->general_steps_host++;
  return BIT1_OK;
}

// Two steps bring the buffer parity and the cell_start swap back to where they were, so a graph of two steps can be
// replayed any number of times.  Returns false when capture is not possible (the caller then launches directly).
static bool build_graph(bit1_ctx* c) {
  const int par = c->cur;
  const uint64_t launches0 = c->launches;
  if (cudaStreamBeginCapture(c->cs, cudaStreamCaptureModeRelaxed) != cudaSuccess) { cudaGetLastError(); return false; }
  enqueue_step(c, nullptr);
  enqueue_step(c, nullptr);
  cudaGraph_t g = nullptr;
  const cudaError_t e = cudaStreamEndCapture(c->cs, &g);
  c->launches = launches0;   // nothing ran yet
  if (e != cudaSuccess || !g) { cudaGetLastError(); return false; }
  cudaGraphExec_t ge = nullptr;
  const cudaError_t e2 = cudaGraphInstantiate(&ge, g, 0);
  cudaGraphDestroy(g);
  if (e2 != cudaSuccess) { cudaGetLastError(); return false; }
  c->graph[par] = ge;
  return true;
}

static bit1_status enqueue_steps(bit1_ctx* c, uint64_t nsteps) {
  if (nsteps && c->ckpt_reads_live) {
    // a checkpoint without staging reads the live half of the store on the side stream: the next step only reads
    // that half too and may overlap the copy; the step after it writes there and has to wait
    enqueue_step(c, nullptr);
    --nsteps;
    CUDA_OK(cudaStreamWaitEvent(c->cs, c->ev_done, 0));
    c->ckpt_reads_live = false;
  }
  if (c->use_graph && !c->profiling && nsteps >= 4) {
    if (!c->graph[c->cur] && !build_graph(c)) c->use_graph = false;
    if (c->graph[c->cur]) {
      const uint64_t per_step = (uint64_t)(c->P.avg_window > 0 ? 5 : 4);
      while (nsteps >= 2) {
        if (cudaGraphLaunch(c->graph[c->cur], c->cs) != cudaSuccess) return BIT1_ERR_CUDA;
        c->launches += 2 * per_step;
        nsteps -= 2;
      }
    }
  }
  for (uint64_t k = 0; k < nsteps; ++k) {
    cudaEvent_t* ev = nullptr;
    if (c->profiling && c->prof_steps < kMaxProfSteps) {
      while (c->prof_ev.size() < (c->prof_steps + 1) * 5) {
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) return BIT1_ERR_CUDA;
        c->prof_ev.push_back(e);
      }
      ev = &c->prof_ev[c->prof_steps * 5];
      c->prof_steps++;
    }
    enqueue_step(c, ev);
  }
  CUDA_OK(cudaGetLastError());
  return BIT1_OK;
}

// Wait for the compute stream and bring the device to step_target: a stalled step (side list beyond its capacity,
// DESIGN.md reading R-side) goes through the general path, the steps enqueued behind it (they returned at once)
// are enqueued again.  After two stalls in a row a growing burst of steps takes the general path outright, so a
// run whose every step overflows does not pay for a wasted mover pass and a host round trip each time.
static bit1_status settle(bit1_ctx* c, DevState* out) {
  DevState h;
  for (;;) {
    BIT1_OK_OR_RETURN(read_state(c, &h));
    if (!h.stalled) break;
    if (h.step >= c->step_target) return BIT1_ERR_CUDA;   // cannot happen: a stall leaves its step undone
    uint64_t left = c->step_target - h.step;              // the stalled step and the no-ops behind it
    if (left & 1ull) flip_parity(c);                      // back to the parity the stalled step found
    c->burst = (c->last_general_step != ~0ull && h.step <= c->last_general_step + 2) ? (c->burst ? 2 * c->burst : 1) : 0;
    if (c->burst > 64) c->burst = 64;
    BIT1_OK_OR_RETURN(enqueue_general_step(c, 0));        // pass A has already counted this step's side effects
    --left;
    uint64_t b = c->burst < left ? c->burst : left;
    left -= b;
    for (; b; --b) BIT1_OK_OR_RETURN(enqueue_general_step(c, 1));
    c->last_general_step = c->step_target - left - 1;
    BIT1_OK_OR_RETURN(enqueue_steps(c, left));
  }
  if (out) *out = h;
  return BIT1_OK;
}

bit1_status bit1_get_profile(bit1_ctx* c, double ms[4], uint64_t* steps) {
  if (!c || !ms) return BIT1_ERR_INVALID_ARG;
  CUDA_OK(cudaStreamSynchronize(c->cs));
  double acc[4] = {0, 0, 0, 0};
  for (size_t k = 0; k < c->prof_steps; ++k)
    for (int j = 0; j < 4; ++j) {
      float t = 0.f;
      CUDA_OK(cudaEventElapsedTime(&t, c->prof_ev[k * 5 + j], c->prof_ev[k * 5 + j + 1]));
      acc[j] += (double)t;
    }
  for (int j = 0; j < 4; ++j) ms[j] = acc[j];
  if (steps) *steps = c->prof_steps;
  c->prof_steps = 0;
  return settle(c, nullptr);
}

// The NEXT-1 settings live in the host-side Params (the launches read them) and ride along in DevState so that a
// checkpoint carries them; clear_sums also zeroes the running and latched averaging sums.
static bit1_status push_settings(bit1_ctx* c, bool clear_sums) {
  drop_graphs(c);
  const int v[4] = {c->P.smooth, c->P.avg_window, c->P.avg_interval, 0};
  CUDA_OK(cudaMemcpyAsync(&c->P.st->smooth_passes, v, sizeof(v), cudaMemcpyHostToDevice, c->cs));
  if (clear_sums) {
    CUDA_OK(cudaMemsetAsync(c->P.acc_dens, 0, avg_bytes(c->P.nc, c->P.ng, c->P.ns), c->cs));
    CUDA_OK(cudaMemsetAsync(&c->P.st->acc_count, 0, 3 * sizeof(unsigned long long), c->cs));
  }
  CUDA_OK(cudaStreamSynchronize(c->cs));   // v is a stack object
  return BIT1_OK;
}

bit1_status bit1_set_recycling(bit1_ctx* c, int species, int to, double vth) {
  if (!c || species < 0 || species >= c->P.ns || to >= c->P.ns || (to >= 0 && !(vth >= 0.0))) return BIT1_ERR_INVALID_ARG;
  if (c->loaded) BIT1_OK_OR_RETURN(settle(c, nullptr));
  drop_graphs(c);
  c->P.sp[species].recycle_to = to < 0 ? -1 : to;
  c->P.sp[species].recycle_vth = to < 0 ? 0.0 : vth;
  rehash(c);
  return BIT1_OK;
}

bit1_status bit1_set_neutral_target(bit1_ctx* c, int species) {
  if (!c || species >= c->P.ns) return BIT1_ERR_INVALID_ARG;
  if (c->loaded) BIT1_OK_OR_RETURN(settle(c, nullptr));
  drop_graphs(c);
  c->P.target_species = species < 0 ? -1 : species;
  c->P.kn = species < 0 ? 0.0
                        : (0.5 * c->weight[species]) / (((double)c->P.sp[species].Q * c->P.area) * c->P.dx);
  rehash(c);
  return BIT1_OK;
}

bit1_status bit1_set_smoothing(bit1_ctx* c, int passes) {
  if (!c || passes < 0 || passes > 8) return BIT1_ERR_INVALID_ARG;
  if (c->loaded) BIT1_OK_OR_RETURN(settle(c, nullptr));   // steps already asked for run with the old setting
  c->P.smooth = passes;
  return push_settings(c, false);
}

bit1_status bit1_set_averaging(bit1_ctx* c, int window, int interval) {
  if (!c || window < 0 || (window > 0 && interval < window)) return BIT1_ERR_INVALID_ARG;
  if (c->loaded) BIT1_OK_OR_RETURN(settle(c, nullptr));
  c->P.avg_window = window;
  c->P.avg_interval = window > 0 ? interval : 0;
  return push_settings(c, true);
}

bit1_status bit1_get_rho_smoothed(bit1_ctx* c, int64_t* out) {
  if (!c || !out) return BIT1_ERR_INVALID_ARG;
  if (!c->loaded) return BIT1_ERR_STATE;
  BIT1_OK_OR_RETURN(settle(c, nullptr));
  CUDA_OK(cudaMemcpyAsync(out, c->P.smooth > 0 ? c->P.rho_s : c->P.rho, (size_t)c->P.ng * 8, cudaMemcpyDeviceToHost, c->cs));
  CUDA_OK(cudaStreamSynchronize(c->cs));
  return BIT1_OK;
}

bit1_status bit1_get_average(bit1_ctx* c, int64_t* dens_sum, double* phi_sum, uint64_t* count, uint64_t* step) {
  if (!c) return BIT1_ERR_INVALID_ARG;
  if (!c->loaded) return BIT1_ERR_STATE;
  DevState h;
  BIT1_OK_OR_RETURN(settle(c, &h));
  if (dens_sum) CUDA_OK(cudaMemcpyAsync(dens_sum, c->P.avg_dens, (size_t)c->P.ns * c->P.ng * 8, cudaMemcpyDeviceToHost, c->cs));
  if (phi_sum) CUDA_OK(cudaMemcpyAsync(phi_sum, c->P.avg_phi, (size_t)(c->P.nc + 1) * 8, cudaMemcpyDeviceToHost, c->cs));
  CUDA_OK(cudaStreamSynchronize(c->cs));
  if (count) *count = h.avg_count;
  if (step) *step = h.avg_step;
  return BIT1_OK;
}

// DevState of a freshly loaded / restarted context: the sort window starts at its smallest radius
static void fresh_window(const Params& P, DevState* h) {
  h->R_cur = P.R_fixed >= 0 ? (unsigned)P.R_fixed : 1u;
  h->R_next = h->R_cur;
  h->stalled = 0;
  for (int e = 0; e < kMaxR + 2; ++e) h->excess[e] = 0;
}

bit1_status bit1_load_particles(bit1_ctx* c, uint64_t n, const double* x, const double* vx, const double* vy,
                                const double* vz, const uint8_t* sp, const uint32_t* pid, int on_device) {
  NvtxRange nvtx_("bit1_load_particles");
  if (!c || (n && (!x || !vx || !vy || !vz || !sp))) return BIT1_ERR_INVALID_ARG;
  if (n > c->P.capacity) return BIT1_ERR_CAPACITY;
  if (c->ckpt_pending) { CUDA_OK(cudaEventSynchronize(c->ev_done)); c->ckpt_pending = false; c->ckpt_reads_live = false; }
  CUDA_OK(cudaStreamSynchronize(c->cs));   // whatever was enqueued (stalled or not) is superseded by the load
  drop_graphs(c);   // the buffer parity restarts at 0 while the cell_start swap keeps its state
  c->loaded = false;
  c->step_target = 0; c->last_general_step = ~0ull; c->burst = 0;
  const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  Particles in = c->buf[1], outp = c->buf[0];
  DevState h0;
  memset(&h0, 0, sizeof(h0));
  fresh_window(c->P, &h0);
  h0.n = (unsigned)n;
  CUDA_OK(cudaMemcpyAsync(c->P.st, &h0, sizeof(DevState), cudaMemcpyHostToDevice, c->cs));
  { bit1_status ps = push_settings(c, true); if (ps != BIT1_OK) return ps; }   // synchronises: h0 is a stack object
  // x, species and pid feed the sort keys and go first on the compute stream; the velocities follow on the side stream
  // while the sort runs and are only needed by its final gather
  const bool split = n && c->ss != c->cs;
  if (n) {
    CUDA_OK(cudaMemcpyAsync(in.x, x, n * 8, kind, c->cs));
    CUDA_OK(cudaMemcpyAsync(in.sp, sp, n, kind, c->cs));
    if (pid) CUDA_OK(cudaMemcpyAsync(in.pid, pid, n * 4, kind, c->cs));
    cudaStream_t vs = split ? c->ss : c->cs;
    if (split) {
      CUDA_OK(cudaEventRecord(c->ev_load0, c->cs));          // everything that used this half of the store is done
      CUDA_OK(cudaStreamWaitEvent(c->ss, c->ev_load0, 0));
    }
    CUDA_OK(cudaMemcpyAsync(in.vx, vx, n * 8, kind, vs));
    if (split) CUDA_OK(cudaEventRecord(c->ev_load1[0], c->ss));
    CUDA_OK(cudaMemcpyAsync(in.vy, vy, n * 8, kind, vs));
    if (split) CUDA_OK(cudaEventRecord(c->ev_load1[1], c->ss));
    CUDA_OK(cudaMemcpyAsync(in.vz, vz, n * 8, kind, vs));
    if (split) CUDA_OK(cudaEventRecord(c->ev_load1[2], c->ss));
  }
  const unsigned n32 = (unsigned)n;
  // validate before anything indexes by species or cell: a bad species tag or a position outside [0, L) is refused
  // here, not carried into the deposit (which would index past the per-species arrays)
  c->launches += launch_load_validate(c->P, in, n32, c->cs);
  DevState h;
  BIT1_OK_OR_RETURN(read_state(c, &h));
  if (h.load_error) {
    if (split) CUDA_OK(cudaStreamSynchronize(c->ss));
    return BIT1_ERR_INVALID_ARG;
  }
  c->launches += launch_load_sort(c->P, in, outp, n32, pid ? 1 : 0, c->ws + c->lay.scratch, c->cs,
                                  split ? c->ev_load1 : nullptr);
  c->cur = 0;
  c->launches += launch_rebuild(c->P, c->buf[0], c->cs);
  CUDA_OK(cudaGetLastError());
  BIT1_OK_OR_RETURN(read_state(c, &h));
  c->loaded = true;
  return BIT1_OK;
}

bit1_status bit1_step(bit1_ctx* c, uint64_t nsteps) {
  NvtxRange nvtx_("bit1_step");
  if (!c) return BIT1_ERR_INVALID_ARG;
  if (!c->loaded) return BIT1_ERR_STATE;
  c->step_target += nsteps;
  return enqueue_steps(c, nsteps);
}

bit1_status bit1_sync(bit1_ctx* c) {
  if (!c) return BIT1_ERR_INVALID_ARG;
  DevState h;
  if (!c->loaded) { BIT1_OK_OR_RETURN(read_state(c, &h)); return BIT1_OK; }
  BIT1_OK_OR_RETURN(settle(c, &h));
  return h.flags ? BIT1_ERR_DEVICE_FLAG : BIT1_OK;
}

static bit1_status fetch(bit1_ctx* c, void* dst, const void* src, size_t bytes) {
  if (!bytes) return BIT1_OK;
  CUDA_OK(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, c->cs));
  return BIT1_OK;
}

bit1_status bit1_get_count(bit1_ctx* c, uint64_t* n_live, uint64_t* step, uint64_t per_species[BIT1_MAX_SPECIES]) {
  if (!c) return BIT1_ERR_INVALID_ARG;
  if (!c->loaded) return BIT1_ERR_STATE;
  if (per_species) {
    bit1_moments m;
    memset(&m, 0, sizeof(m));
    bit1_status s = bit1_get_moments(c, &m);
    if (s != BIT1_OK) return s;
    for (int k = 0; k < BIT1_MAX_SPECIES; ++k) per_species[k] = m.count[k];
    if (n_live) *n_live = m.n_live;
    if (step) *step = m.step;
    return BIT1_OK;
  }
  DevState h;
  BIT1_OK_OR_RETURN(settle(c, &h));
  if (n_live) *n_live = h.n;
  if (step) *step = h.step;
  return BIT1_OK;
}

bit1_status bit1_get_rho(bit1_ctx* c, int64_t* rho_fixed, double* rho_si) {
  if (!c) return BIT1_ERR_INVALID_ARG;
  if (!c->loaded) return BIT1_ERR_STATE;
  BIT1_OK_OR_RETURN(settle(c, nullptr));
  const int ng = c->P.ng;
  int64_t* tmp = rho_fixed;
  if (!tmp) tmp = static_cast<int64_t*>(malloc((size_t)ng * 8));
  if (!tmp) return BIT1_ERR_INVALID_ARG;
  bit1_status s = fetch(c, tmp, c->P.rho, (size_t)ng * 8);
  if (s == BIT1_OK && cudaStreamSynchronize(c->cs) != cudaSuccess) s = BIT1_ERR_CUDA;
  if (s == BIT1_OK && rho_si) {
    const double f = kTwoM40 / (c->P.area * c->P.dx);
    for (int j = 0; j < ng; ++j) {
      double v = (double)tmp[j] * f;
      if (c->P.bc && (j == 0 || j == c->P.nc)) v = 2.0 * v;
      rho_si[j] = v;
    }
  }
  if (!rho_fixed) free(tmp);
  return s;
}

bit1_status bit1_get_phi(bit1_ctx* c, double* phi) {
  if (!c || !phi) return BIT1_ERR_INVALID_ARG;
  if (!c->loaded) return BIT1_ERR_STATE;
  BIT1_OK_OR_RETURN(settle(c, nullptr));
  BIT1_OK_OR_RETURN(fetch(c, phi, c->P.phi, (size_t)(c->P.nc + 1) * 8));
  CUDA_OK(cudaStreamSynchronize(c->cs));
  return BIT1_OK;
}

bit1_status bit1_get_E(bit1_ctx* c, double* E) {
  if (!c || !E) return BIT1_ERR_INVALID_ARG;
  if (!c->loaded) return BIT1_ERR_STATE;
  BIT1_OK_OR_RETURN(settle(c, nullptr));
  BIT1_OK_OR_RETURN(fetch(c, E, c->P.E, (size_t)(c->P.nc + 1) * 8));
  CUDA_OK(cudaStreamSynchronize(c->cs));
  return BIT1_OK;
}

bit1_status bit1_get_dens(bit1_ctx* c, int64_t* dens) {
  if (!c || !dens) return BIT1_ERR_INVALID_ARG;
  if (!c->loaded) return BIT1_ERR_STATE;
  BIT1_OK_OR_RETURN(settle(c, nullptr));
  BIT1_OK_OR_RETURN(fetch(c, dens, c->P.dens, (size_t)c->P.ns * c->P.ng * 8));
  CUDA_OK(cudaStreamSynchronize(c->cs));
  return BIT1_OK;
}

bit1_status bit1_get_moments(bit1_ctx* c, bit1_moments* out) {
  NvtxRange nvtx_("bit1_get_moments");
  if (!c || !out) return BIT1_ERR_INVALID_ARG;
  if (!c->loaded) return BIT1_ERR_STATE;
  BIT1_OK_OR_RETURN(settle(c, nullptr));
  const Params& P = c->P;
  double* partial = reinterpret_cast<double*>(c->ws + c->lay.mom);
  double* dres = partial + (size_t)1024 * kMaxSpecies * 3;
  c->launches += launch_moments(P, c->buf[c->cur], partial, dres, c->cs);
  double res[kMaxSpecies * 3 + 1];
  CUDA_OK(cudaMemcpyAsync(res, dres, sizeof(res), cudaMemcpyDeviceToHost, c->cs));
  DevState h;
  bit1_status s = read_state(c, &h);
  if (s != BIT1_OK) return s;
  double* dens_out[BIT1_MAX_SPECIES];
  for (int k = 0; k < BIT1_MAX_SPECIES; ++k) dens_out[k] = out->density[k];
  out->step = h.step; out->n_live = h.n;
  for (int k = 0; k < BIT1_MAX_SPECIES; ++k) {
    out->count[k] = 0; out->kinetic_J[k] = 0.0; out->px[k] = 0.0; out->candidates[k] = h.candidates[k];
    for (int e = 0; e < 3; ++e) out->events[k][e] = h.events[k][e];
    out->wall_count[0][k] = h.wall_count[0][k];
    out->wall_count[1][k] = h.wall_count[1][k];
  }
  for (int k = 0; k < P.ns; ++k) {
    out->count[k] = (uint64_t)res[k * 3];
    out->kinetic_J[k] = ((0.5 * c->m[k]) * c->weight[k]) * res[k * 3 + 1];
    out->px[k] = (c->m[k] * c->weight[k]) * res[k * 3 + 2];
  }
  out->field_J = P.field_J_factor * res[kMaxSpecies * 3];
  out->wall_charge_fixed[0] = h.wall_charge[0];
  out->wall_charge_fixed[1] = h.wall_charge[1];
  out->rho_total_fixed = h.rho_total;
  out->flags = h.flags; out->next_pid = h.next_pid;
  out->nu_overflow = h.nu_overflow; out->dir_fallback = h.dir_fallback; out->escape = h.escape;
  out->births = h.births; out->reinject = h.reinject; out->recycled = h.recycled;
  out->far_movers = h.far_movers; out->max_far_movers_per_step = h.max_far_movers;
  out->general_steps = h.general_steps; out->window_radius = h.R_cur;
  out->check_failures = h.check_count; out->check_line = h.check_line; out->_pad = 0;
  out->check_index = h.check_idx; out->check_limit = h.check_limit;
  bool any = false;
  for (int k = 0; k < P.ns; ++k) any = any || dens_out[k];
  if (any) {
    const size_t ng = (size_t)P.ng;
    int64_t* tmp = static_cast<int64_t*>(malloc((size_t)P.ns * ng * 8));
    if (!tmp) return BIT1_ERR_INVALID_ARG;
    s = bit1_get_dens(c, tmp);
    if (s == BIT1_OK) {
      for (int k = 0; k < P.ns; ++k) {
        if (!dens_out[k]) continue;
        for (size_t j = 0; j < ng; ++j) {
          double v = (((double)tmp[k * ng + j] / (double)P.sp[k].Q) * c->weight[k]) / (P.area * P.dx);
          if (P.bc && (j == 0 || j == (size_t)P.nc)) v = 2.0 * v;
          dens_out[k][j] = v;
        }
      }
    }
    free(tmp);
    if (s != BIT1_OK) return s;
  }
  return BIT1_OK;
}

bit1_status bit1_get_particles(bit1_ctx* c, double* x, double* vx, double* vy, double* vz, int32_t* cell,
                               uint32_t* pid, uint8_t* sp, int64_t* cell_start) {
  if (!c) return BIT1_ERR_INVALID_ARG;
  if (!c->loaded) return BIT1_ERR_STATE;
  DevState h;
  BIT1_OK_OR_RETURN(settle(c, &h));
  const size_t n = h.n;
  const Particles& p = c->buf[c->cur];
  if (x) CUDA_OK(cudaMemcpyAsync(x, p.x, n * 8, cudaMemcpyDeviceToHost, c->cs));
  if (vx) CUDA_OK(cudaMemcpyAsync(vx, p.vx, n * 8, cudaMemcpyDeviceToHost, c->cs));
  if (vy) CUDA_OK(cudaMemcpyAsync(vy, p.vy, n * 8, cudaMemcpyDeviceToHost, c->cs));
  if (vz) CUDA_OK(cudaMemcpyAsync(vz, p.vz, n * 8, cudaMemcpyDeviceToHost, c->cs));
  if (cell) {
    // the store's cell index is cell_of(x) by construction; no step reads or writes the array, it is filled on demand
    c->launches += launch_fill_cells(c->P, p, c->cs);
    CUDA_OK(cudaMemcpyAsync(cell, p.cell, n * 4, cudaMemcpyDeviceToHost, c->cs));
  }
  if (pid) CUDA_OK(cudaMemcpyAsync(pid, p.pid, n * 4, cudaMemcpyDeviceToHost, c->cs));
  if (sp) CUDA_OK(cudaMemcpyAsync(sp, p.sp, n, cudaMemcpyDeviceToHost, c->cs));
  int32_t* cs32 = nullptr;
  if (cell_start) {
    cs32 = static_cast<int32_t*>(malloc((size_t)(c->P.nc + 1) * 4));
    if (!cs32) return BIT1_ERR_INVALID_ARG;
    if (cudaMemcpyAsync(cs32, c->P.cell_start, (size_t)(c->P.nc + 1) * 4, cudaMemcpyDeviceToHost, c->cs) != cudaSuccess) {
      free(cs32);
      return BIT1_ERR_CUDA;
    }
  }
  cudaError_t e = cudaStreamSynchronize(c->cs);
  if (cs32) {
    if (e == cudaSuccess) for (int j = 0; j <= c->P.nc; ++j) cell_start[j] = cs32[j];
    free(cs32);
  }
  return e == cudaSuccess ? BIT1_OK : BIT1_ERR_CUDA;
}

bit1_status bit1_export_species(bit1_ctx* c, int species, uint64_t capacity_out, uint64_t* n_out,
                                int64_t* counts_per_cell, double* x, double* vx, double* vy, double* vz,
                                uint32_t* pid) {
  if (!c || species < 0 || species >= c->P.ns || !n_out) return BIT1_ERR_INVALID_ARG;
  if (!c->loaded) return BIT1_ERR_STATE;
  BIT1_OK_OR_RETURN(settle(c, nullptr));
  // a checkpoint without staging may still be reading the store; the idle half is about to be written
  if (c->ckpt_pending) { CUDA_OK(cudaEventSynchronize(c->ev_done)); c->ckpt_pending = false; c->ckpt_reads_live = false; }
  char* sc = c->ws + c->lay.exp;
  c->launches += launch_export_count(c->P, c->buf[c->cur], species, c->P.capacity, sc, c->cs);
  unsigned long long total = 0;
  CUDA_OK(cudaMemcpyAsync(&total, sc, 8, cudaMemcpyDeviceToHost, c->cs));
  CUDA_OK(cudaStreamSynchronize(c->cs));
  *n_out = total;
  if (counts_per_cell) {
    int32_t* tmp = static_cast<int32_t*>(malloc((size_t)c->P.nc * 4));
    if (!tmp) return BIT1_ERR_INVALID_ARG;
    cudaError_t e = cudaMemcpyAsync(tmp, sc + 256, (size_t)c->P.nc * 4, cudaMemcpyDeviceToHost, c->cs);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->cs);
    if (e == cudaSuccess) for (int j = 0; j < c->P.nc; ++j) counts_per_cell[j] = tmp[j];
    free(tmp);
    if (e != cudaSuccess) return BIT1_ERR_CUDA;
  }
  if (!x && !vx && !vy && !vz && !pid) return BIT1_OK;   // size query
  if (capacity_out < total) return BIT1_ERR_CAPACITY;
  // the other particle buffer is free between steps: the records are compacted into it, then copied out
  const Particles& out = c->buf[c->cur ^ 1];
  c->launches += launch_export_scatter(c->P, c->buf[c->cur], out, species, sc, c->cs);
  const size_t n = (size_t)total;
  if (x) CUDA_OK(cudaMemcpyAsync(x, out.x, n * 8, cudaMemcpyDeviceToHost, c->cs));
  if (vx) CUDA_OK(cudaMemcpyAsync(vx, out.vx, n * 8, cudaMemcpyDeviceToHost, c->cs));
  if (vy) CUDA_OK(cudaMemcpyAsync(vy, out.vy, n * 8, cudaMemcpyDeviceToHost, c->cs));
  if (vz) CUDA_OK(cudaMemcpyAsync(vz, out.vz, n * 8, cudaMemcpyDeviceToHost, c->cs));
  if (pid) CUDA_OK(cudaMemcpyAsync(pid, out.pid, n * 4, cudaMemcpyDeviceToHost, c->cs));
  CUDA_OK(cudaStreamSynchronize(c->cs));
  CUDA_OK(cudaGetLastError());
  return BIT1_OK;
}

bit1_status bit1_set_E(bit1_ctx* c, const double* E, int freeze) {
  if (!c || !E) return BIT1_ERR_INVALID_ARG;
  if (!c->loaded) return BIT1_ERR_STATE;
  BIT1_OK_OR_RETURN(settle(c, nullptr));
  CUDA_OK(cudaMemcpyAsync(c->P.E, E, (size_t)(c->P.nc + 1) * 8, cudaMemcpyHostToDevice, c->cs));
  const unsigned f = freeze ? 1u : 0u;
  CUDA_OK(cudaMemcpyAsync(&c->P.st->freeze_field, &f, 4, cudaMemcpyHostToDevice, c->cs));
  CUDA_OK(cudaStreamSynchronize(c->cs));
  return BIT1_OK;
}

bit1_status bit1_set_step(bit1_ctx* c, uint64_t step) {
  if (!c) return BIT1_ERR_INVALID_ARG;
  if (!c->loaded) return BIT1_ERR_STATE;
  BIT1_OK_OR_RETURN(settle(c, nullptr));
  CUDA_OK(cudaMemcpyAsync(&c->P.st->step, &step, 8, cudaMemcpyHostToDevice, c->cs));
  CUDA_OK(cudaStreamSynchronize(c->cs));
  c->step_target = step;
  c->last_general_step = ~0ull;
  return BIT1_OK;
}

size_t bit1_checkpoint_size(bit1_ctx* c) {
  if (!c) return 0;
  return ckpt_layout(c->P.nc, c->P.ng, c->P.ns, c->P.capacity).bytes;
}

bit1_status bit1_checkpoint(bit1_ctx* c, void* host, size_t cap, size_t* written) {
  NvtxRange nvtx_("bit1_checkpoint");
  if (!c || !host) return BIT1_ERR_INVALID_ARG;
  if (!c->loaded) return BIT1_ERR_STATE;
  if (c->ckpt_pending) { CUDA_OK(cudaEventSynchronize(c->ev_done)); c->ckpt_pending = false; c->ckpt_reads_live = false; }
  // the live particle count sizes the blob, so the steps asked for so far are waited for here; the copy itself
  // (the expensive part) runs on the side stream behind an event and overlaps the steps that follow
  DevState h;
  BIT1_OK_OR_RETURN(settle(c, &h));
  // The blob holds no E: bit1_restart rebuilds the field from rho.  Under a prescribed, frozen field (bit1_set_E with
  // freeze_field) that rebuild would silently swap the caller's field for the self-consistent one, and the restarted
  // run would no longer be the run that was saved.  Refuse rather than write a checkpoint that cannot keep the promise.
  if (h.freeze_field) return BIT1_ERR_STATE;
  const size_t n = h.n;
  const CkptLayout cl = ckpt_layout(c->P.nc, c->P.ng, c->P.ns, n);
  if (cap < cl.bytes) return BIT1_ERR_CAPACITY;
  CkptHeader hd;
  memset(&hd, 0, sizeof(hd));
  memcpy(hd.magic, "BIT1CKPT", 8);
  hd.version = kCkptVersion; hd.nc = c->P.nc; hd.ns = c->P.ns; hd.bc = c->P.bc;
  hd.capacity = c->P.capacity; hd.cfg_hash = c->cfg_hash; hd.bytes = cl.bytes; hd.n = n;
  memset(host, 0, 256);
  memcpy(host, &hd, sizeof(hd));
  char* hb = static_cast<char*>(host);
  const Particles& p = c->buf[c->cur];
  const size_t ab = avg_bytes(c->P.nc, c->P.ng, c->P.ns);
  const cudaMemcpyKind d2d = cudaMemcpyDeviceToDevice, d2h = cudaMemcpyDeviceToHost;
  if (c->staging) {
    // snapshot on the compute stream (blob layout, live particles only), one copy out on the side stream: the
    // steps that follow overlap the D2H and are free to overwrite the store
    char* sg = c->ws + c->lay.scratch;
    CUDA_OK(cudaMemcpyAsync(sg + cl.state, c->P.st, sizeof(DevState), d2d, c->cs));
    CUDA_OK(cudaMemcpyAsync(sg + cl.avg, c->P.acc_dens, ab, d2d, c->cs));
    if (n) {
      CUDA_OK(cudaMemcpyAsync(sg + cl.x, p.x, n * 8, d2d, c->cs));
      CUDA_OK(cudaMemcpyAsync(sg + cl.vx, p.vx, n * 8, d2d, c->cs));
      CUDA_OK(cudaMemcpyAsync(sg + cl.vy, p.vy, n * 8, d2d, c->cs));
      CUDA_OK(cudaMemcpyAsync(sg + cl.vz, p.vz, n * 8, d2d, c->cs));
      CUDA_OK(cudaMemcpyAsync(sg + cl.pid, p.pid, n * 4, d2d, c->cs));
      CUDA_OK(cudaMemcpyAsync(sg + cl.sp, p.sp, n, d2d, c->cs));
    }
    CUDA_OK(cudaEventRecord(c->ev_snap, c->cs));
    CUDA_OK(cudaStreamWaitEvent(c->ss, c->ev_snap, 0));
    CUDA_OK(cudaMemcpyAsync(hb + cl.state, sg + cl.state, cl.bytes - cl.state, d2h, c->ss));
    CUDA_OK(cudaEventRecord(c->ev_done, c->ss));
  } else {
    // no snapshot area: the small mutable pieces are snapshotted, the particle arrays are copied out of the live
    // half of the store on the side stream; the next step only reads that half and may overlap, the one after
    // waits for the copy (enqueue_steps)
    char* sm = c->ws + c->lay.small;
    const CkptLayout c0 = ckpt_layout(c->P.nc, c->P.ng, c->P.ns, 0);
    CUDA_OK(cudaMemcpyAsync(sm + c0.state, c->P.st, sizeof(DevState), d2d, c->cs));
    CUDA_OK(cudaMemcpyAsync(sm + c0.avg, c->P.acc_dens, ab, d2d, c->cs));
    CUDA_OK(cudaEventRecord(c->ev_snap, c->cs));
    CUDA_OK(cudaStreamWaitEvent(c->ss, c->ev_snap, 0));
    CUDA_OK(cudaMemcpyAsync(hb + cl.state, sm + c0.state, sizeof(DevState), d2h, c->ss));
    CUDA_OK(cudaMemcpyAsync(hb + cl.avg, sm + c0.avg, ab, d2h, c->ss));
    if (n) {
      CUDA_OK(cudaMemcpyAsync(hb + cl.x, p.x, n * 8, d2h, c->ss));
      CUDA_OK(cudaMemcpyAsync(hb + cl.vx, p.vx, n * 8, d2h, c->ss));
      CUDA_OK(cudaMemcpyAsync(hb + cl.vy, p.vy, n * 8, d2h, c->ss));
      CUDA_OK(cudaMemcpyAsync(hb + cl.vz, p.vz, n * 8, d2h, c->ss));
      CUDA_OK(cudaMemcpyAsync(hb + cl.pid, p.pid, n * 4, d2h, c->ss));
      CUDA_OK(cudaMemcpyAsync(hb + cl.sp, p.sp, n, d2h, c->ss));
    }
    CUDA_OK(cudaEventRecord(c->ev_done, c->ss));
    c->ckpt_reads_live = c->ss != c->cs;
  }
  c->ckpt_pending = true;
  if (written) *written = cl.bytes;
  return BIT1_OK;
}

bit1_status bit1_checkpoint_wait(bit1_ctx* c) {
  if (!c) return BIT1_ERR_INVALID_ARG;
  if (c->ckpt_pending) {
    CUDA_OK(cudaEventSynchronize(c->ev_done));
    c->ckpt_pending = false;
    c->ckpt_reads_live = false;
  }
  return BIT1_OK;
}

bit1_status bit1_restart(bit1_ctx* c, const void* blob, size_t bytes) {
  NvtxRange nvtx_("bit1_restart");
  if (!c || !blob) return BIT1_ERR_INVALID_ARG;
  if (bytes < 256 + sizeof(DevState)) return BIT1_ERR_CHECKPOINT;
  CkptHeader hd;
  memcpy(&hd, blob, sizeof(hd));
  if (memcmp(hd.magic, "BIT1CKPT", 8) != 0 || hd.version != kCkptVersion || hd.nc != c->P.nc || hd.ns != c->P.ns ||
      hd.bc != c->P.bc || hd.capacity != c->P.capacity || hd.cfg_hash != c->cfg_hash || hd.n > c->P.capacity)
    return BIT1_ERR_CHECKPOINT;
  const size_t n = (size_t)hd.n;
  const CkptLayout cl = ckpt_layout(c->P.nc, c->P.ng, c->P.ns, n);
  if (hd.bytes != cl.bytes || bytes < cl.bytes) return BIT1_ERR_CHECKPOINT;
  if (c->ckpt_pending) { CUDA_OK(cudaEventSynchronize(c->ev_done)); c->ckpt_pending = false; c->ckpt_reads_live = false; }
  drop_graphs(c);
  const char* hb = static_cast<const char*>(blob);
  DevState h;
  memcpy(&h, hb + cl.state, sizeof(DevState));
  if (h.n != n) return BIT1_ERR_CHECKPOINT;
  h.ovf_count = 0; h.ovf_valid = 0; h.freeze_field = 0; h.load_error = 0; h.n_next = h.n;
  fresh_window(c->P, &h);
  CUDA_OK(cudaStreamSynchronize(c->cs));
  if (h.smooth_passes < 0 || h.smooth_passes > 8 || h.avg_window < 0 || h.avg_interval < h.avg_window)
    return BIT1_ERR_CHECKPOINT;
  c->loaded = false;
  CUDA_OK(cudaMemcpyAsync(c->P.st, &h, sizeof(DevState), cudaMemcpyHostToDevice, c->cs));
  CUDA_OK(cudaStreamSynchronize(c->cs));  // h is a stack object
  c->P.smooth = h.smooth_passes; c->P.avg_window = h.avg_window; c->P.avg_interval = h.avg_interval;
  CUDA_OK(cudaMemcpyAsync(c->P.acc_dens, hb + cl.avg, avg_bytes(c->P.nc, c->P.ng, c->P.ns), cudaMemcpyHostToDevice, c->cs));
  c->cur = 0;
  const Particles& p = c->buf[0];
  const cudaMemcpyKind h2d = cudaMemcpyHostToDevice;
  if (n) {
    CUDA_OK(cudaMemcpyAsync(p.x, hb + cl.x, n * 8, h2d, c->cs));
    CUDA_OK(cudaMemcpyAsync(p.vx, hb + cl.vx, n * 8, h2d, c->cs));
    CUDA_OK(cudaMemcpyAsync(p.vy, hb + cl.vy, n * 8, h2d, c->cs));
    CUDA_OK(cudaMemcpyAsync(p.vz, hb + cl.vz, n * 8, h2d, c->cs));
    CUDA_OK(cudaMemcpyAsync(p.pid, hb + cl.pid, n * 4, h2d, c->cs));
    CUDA_OK(cudaMemcpyAsync(p.sp, hb + cl.sp, n, h2d, c->cs));
  }
  // the blob's body is data from outside: species tags, positions and their order are checked before anything
  // indexes by them (header and hash only vouch for the configuration)
  c->launches += launch_state_validate(c->P, p, (unsigned)n, c->cs);
  DevState hv;
  BIT1_OK_OR_RETURN(read_state(c, &hv));
  if (hv.load_error) return BIT1_ERR_CHECKPOINT;
  c->launches += launch_rebuild(c->P, c->buf[0], c->cs);
  CUDA_OK(cudaGetLastError());
  CUDA_OK(cudaStreamSynchronize(c->cs));
  c->step_target = h.step; c->last_general_step = ~0ull; c->burst = 0;
  c->loaded = true;
  return BIT1_OK;
}

// ---- streaming checkpoints (second half) -------------------------------------------------
static void CUDART_CB stream_done_cb(void* p) {
  // runs on a CUDA-internal thread once the side-stream copy into the slot has landed: publish the sequence number
  bit1_ctx::StreamDone* d = static_cast<bit1_ctx::StreamDone*>(p);
  bit1_ctx* c = d->c;
  bit1_stream_header* hd = reinterpret_cast<bit1_stream_header*>(c->ring + (size_t)d->slot * c->slot_bytes);
  std::atomic_thread_fence(std::memory_order_release);
  reinterpret_cast<std::atomic<uint64_t>*>(&hd->seq)->store(d->seq, std::memory_order_release);
  c->slot_seq[d->slot].store(d->seq, std::memory_order_release);
  c->slot_state[d->slot].store(kSlotReady, std::memory_order_release);
}

size_t bit1_stream_slot_size(bit1_ctx* c) {
  if (!c) return 0;
  return sizeof(bit1_stream_header) + stream_payload_bytes(c->P.nc, c->P.ns, c->P.capacity);
}

bit1_status bit1_stream_open(bit1_ctx* c, void* ring, size_t slot_bytes, int nslots) {
  if (!c || !ring || nslots < 2 || nslots > BIT1_STREAM_MAX_SLOTS || (slot_bytes & (kAlign - 1)) ||
      (reinterpret_cast<uintptr_t>(ring) & (kAlign - 1)))
    return BIT1_ERR_INVALID_ARG;
  if (!c->staging || c->ss == c->cs) return BIT1_ERR_STATE;   // needs the device snapshot area and a side stream
  if (c->ring) return BIT1_ERR_STATE;
  if (slot_bytes < sizeof(bit1_stream_header) + 5 * kAlign) return BIT1_ERR_CAPACITY;
  c->ring = static_cast<char*>(ring);
  c->slot_bytes = slot_bytes;
  c->nslots = nslots;
  for (int k = 0; k < nslots; ++k) {
    c->slot_state[k].store(kSlotFree);
    c->slot_seq[k].store(0);
    memset(c->ring + (size_t)k * slot_bytes, 0, sizeof(bit1_stream_header));
  }
  return BIT1_OK;
}

bit1_status bit1_stream_close(bit1_ctx* c) {
  if (!c) return BIT1_ERR_INVALID_ARG;
  if (c->ckpt_pending) { CUDA_OK(cudaEventSynchronize(c->ev_done)); c->ckpt_pending = false; c->ckpt_reads_live = false; }
  if (c->ss != c->cs) CUDA_OK(cudaStreamSynchronize(c->ss));   // the host function has run
  c->ring = nullptr; c->nslots = 0;
  return BIT1_OK;
}

bit1_status bit1_stream_publish(bit1_ctx* c, uint64_t* seq_out) {
  NvtxRange nvtx_("bit1_stream_publish");
  if (!c) return BIT1_ERR_INVALID_ARG;
  if (!c->loaded || !c->ring) return BIT1_ERR_STATE;
  // one snapshot in flight at a time: the device staging area is shared with bit1_checkpoint
  if (c->ckpt_pending) { CUDA_OK(cudaEventSynchronize(c->ev_done)); c->ckpt_pending = false; c->ckpt_reads_live = false; }
  DevState h;
  BIT1_OK_OR_RETURN(settle(c, &h));
  // a slot the consumer does not hold: a free one, else the oldest unread one (it is dropped, as a bounded SST queue does)
  int slot = -1;
  uint64_t oldest = ~0ull;
  for (int k = 0; k < c->nslots && slot < 0; ++k)
    if (c->slot_state[k].load(std::memory_order_acquire) == kSlotFree) slot = k;
  if (slot < 0) {
    for (int k = 0; k < c->nslots; ++k)
      if (c->slot_state[k].load(std::memory_order_acquire) == kSlotReady && c->slot_seq[k].load() < oldest) {
        oldest = c->slot_seq[k].load();
        slot = k;
      }
    if (slot >= 0) {
      int expect = kSlotReady;   // the consumer may grab it at this very moment: then it is held, look no further
      if (!c->slot_state[slot].compare_exchange_strong(expect, kSlotFilling)) slot = -1;
    }
  } else {
    c->slot_state[slot].store(kSlotFilling, std::memory_order_release);
  }
  if (slot < 0) return BIT1_ERR_CAPACITY;   // every slot is held by the consumer
  // a failure below (a CUDA error, a slot too small) hands the claimed slot back instead of leaving it "filling" for good
  struct SlotClaim {
    std::atomic<int>* state;
    bool armed;
    ~SlotClaim() { if (armed) state->store(kSlotFree, std::memory_order_release); }
  } claim{&c->slot_state[slot], true};
  const Params& P = c->P;
  const int nc = P.nc, ns = P.ns;
  char* sg = c->ws + c->lay.scratch;   // device staging, payload layout (offsets relative to the end of the header)
  char* ex = c->ws + c->lay.exp;
  bit1_stream_header hd;
  memset(&hd, 0, sizeof(hd));
  memcpy(hd.magic, "BIT1STRM", 8);
  const uint64_t seq = c->next_seq++;
  hd.seq_begin = seq; hd.seq = 0; hd.step = h.step; hd.n_total = h.n; hd.nc = nc; hd.ns = ns; hd.bc = P.bc;
  size_t o = 0;
  const size_t hsz = sizeof(bit1_stream_header);
  for (int s = 0; s < ns; ++s) {
    // counts per cell and the species' total ("the vector of particle counts per cell", then the records)
    c->launches += launch_export_count(P, c->buf[c->cur], s, P.capacity, ex, c->cs);
    unsigned long long total = 0;
    CUDA_OK(cudaMemcpyAsync(&total, ex, 8, cudaMemcpyDeviceToHost, c->cs));
    CUDA_OK(cudaStreamSynchronize(c->cs));
    const size_t n = (size_t)total;
    hd.count[s] = total;
    hd.off_counts[s] = hsz + o; o += align_up((size_t)nc * 4);
    hd.off_x[s] = hsz + o; o += align_up(n * 8);
    hd.off_vx[s] = hsz + o; o += align_up(n * 8);
    hd.off_vy[s] = hsz + o; o += align_up(n * 8);
    hd.off_vz[s] = hsz + o; o += align_up(n * 8);
    hd.off_pid[s] = hsz + o; o += align_up(n * 4);
    if (hsz + o > c->slot_bytes) return BIT1_ERR_CAPACITY;
    CUDA_OK(cudaMemcpyAsync(sg + (hd.off_counts[s] - hsz), ex + 256, (size_t)nc * 4, cudaMemcpyDeviceToDevice, c->cs));
    Particles out;
    memset(&out, 0, sizeof(out));
    out.x = reinterpret_cast<double*>(sg + (hd.off_x[s] - hsz));
    out.vx = reinterpret_cast<double*>(sg + (hd.off_vx[s] - hsz));
    out.vy = reinterpret_cast<double*>(sg + (hd.off_vy[s] - hsz));
    out.vz = reinterpret_cast<double*>(sg + (hd.off_vz[s] - hsz));
    out.pid = reinterpret_cast<unsigned*>(sg + (hd.off_pid[s] - hsz));
    if (n) c->launches += launch_export_scatter(P, c->buf[c->cur], out, s, ex, c->cs);
  }
  hd.bytes = hsz + o;
  char* hs = c->ring + (size_t)slot * c->slot_bytes;
  // a reader in another process sees seq != seq_begin while the slot is being filled
  memcpy(hs, &hd, sizeof(hd));
  std::atomic_thread_fence(std::memory_order_release);
  CUDA_OK(cudaEventRecord(c->ev_snap, c->cs));
  CUDA_OK(cudaStreamWaitEvent(c->ss, c->ev_snap, 0));
  if (o) CUDA_OK(cudaMemcpyAsync(hs + hsz, sg, o, cudaMemcpyDeviceToHost, c->ss));
  c->done_arg[slot].c = c; c->done_arg[slot].slot = slot; c->done_arg[slot].seq = seq;
  CUDA_OK(cudaLaunchHostFunc(c->ss, stream_done_cb, &c->done_arg[slot]));
  claim.armed = false;   // from here on the host function publishes the slot
  CUDA_OK(cudaEventRecord(c->ev_done, c->ss));
  c->ckpt_pending = true;
  if (seq_out) *seq_out = seq;
  return BIT1_OK;
}

bit1_status bit1_stream_acquire(bit1_ctx* c, uint64_t after_seq, const void** slot_out, uint64_t* seq_out) {
  if (!c || !slot_out || !seq_out) return BIT1_ERR_INVALID_ARG;
  if (!c->ring) return BIT1_ERR_STATE;
  for (;;) {
    int best = -1;
    uint64_t bs = after_seq;
    for (int k = 0; k < c->nslots; ++k) {
      if (c->slot_state[k].load(std::memory_order_acquire) != kSlotReady) continue;
      const uint64_t q = c->slot_seq[k].load(std::memory_order_acquire);
      if (q > bs) { bs = q; best = k; }
    }
    if (best < 0) return BIT1_ERR_STATE;   // nothing newer than after_seq yet
    int expect = kSlotReady;
    if (c->slot_state[best].compare_exchange_strong(expect, kSlotHeld, std::memory_order_acq_rel)) {
      // The slot is ours now and the producer keeps off it, so its sequence number can no longer change.  Read it
      // again: between the scan above and the exchange the producer may have reclaimed the slot and published a newer
      // snapshot into it (state Ready again, so the exchange still succeeded).  What the slot holds is then that newer
      // snapshot, complete (the number is stored before the state), and its number is the one bit1_stream_release
      // will be given -- the number seen by the scan would match no slot and the slot would stay held for good.
      const uint64_t now = c->slot_seq[best].load(std::memory_order_acquire);
      if (now <= after_seq) {   // cannot happen with increasing numbers; never hand out what the caller has seen
        c->slot_state[best].store(kSlotReady, std::memory_order_release);
        continue;
      }
      *slot_out = c->ring + (size_t)best * c->slot_bytes;
      *seq_out = now;
      return BIT1_OK;
    }
    // the producer took it back for the next snapshot in the meantime: look again
  }
}

bit1_status bit1_stream_release(bit1_ctx* c, uint64_t seq) {
  if (!c) return BIT1_ERR_INVALID_ARG;
  if (!c->ring) return BIT1_ERR_STATE;
  for (int k = 0; k < c->nslots; ++k)
    if (c->slot_state[k].load(std::memory_order_acquire) == kSlotHeld && c->slot_seq[k].load() == seq) {
      c->slot_state[k].store(kSlotFree, std::memory_order_release);
      return BIT1_OK;
    }
  return BIT1_ERR_INVALID_ARG;
}

}  // extern "C"
