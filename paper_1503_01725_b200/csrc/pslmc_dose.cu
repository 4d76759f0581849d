// pslmc_dose.cu — the batching driver and the C ABI of the hot path: iterated k_sample → k_photon /
// k_electron launches per sub-source type and energy order, secondary
// queues, int64 scoring, finalise, stats.  No CPU fallback: every entry point here needs a device.
#include "pslmc_host.h"
#include "pslmc_transport.cuh"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>

namespace pslmc {

#define CUDA_TRY(expr)                                                                         \
  do {                                                                                         \
    cudaError_t e_ = (expr);                                                                   \
    if (e_ != cudaSuccess) {                                                                   \
      char b_[512];                                                                            \
      snprintf(b_, sizeof b_, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__, __LINE__); \
      return fail(MC_E_CUDA, b_);                                                              \
    }                                                                                          \
  } while (0)

thread_local mc_stats_t g_stats;

// Library-managed scratch (used when the caller passes no workspace).  One per process; calls are
// not re-entrant (see pslmc.h).
struct Scratch { void *ptr = nullptr; size_t bytes = 0; };
static Scratch g_scratch, g_hostio;

static int scratch_get(Scratch &s, size_t bytes, void **out) {
  if (s.bytes < bytes) {
    if (s.ptr) cudaFree(s.ptr);
    s.ptr = nullptr; s.bytes = 0;
    CUDA_TRY(cudaMalloc(&s.ptr, bytes));
    s.bytes = bytes;
  }
  *out = s.ptr;
  return MC_OK;
}

static size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

// Workspace layout for a batch of B primaries.  Shared by the whole call: group offsets, cross-section
// data, packed phantom, (optionally) the int64 dose grid.  Per pipeline (kMaxPipes of them, see run_dose):
// control block, the particle buffer (2 planes + the commissioning column), the electron queue (capacity 4B, 3 planes).
constexpr int kMaxPipes = 2;
struct Layout {
  size_t ctl, off, xs, vox, p0, p1, p2, eq[3], acc, total;
  unsigned eq_cap;
};
static void make_layouts(uint64_t batch, size_t nvox, bool with_acc, Layout out[kMaxPipes]) {
  Layout L; size_t o = 0;
  auto take = [&](size_t b) { size_t at = o; o += align_up(b); return at; };
  L.eq_cap = (unsigned)std::min<uint64_t>(4 * batch, 0x7fffffffu);
  if (const char *e = getenv("PSLMC_TEST_EQ_CAP")) L.eq_cap = (unsigned)std::max(1, atoi(e));   // test hook: exercises MC_E_OVERFLOW (the planes keep their full size)
  size_t ctl_at[kMaxPipes];
  for (int p = 0; p < kMaxPipes; ++p) ctl_at[p] = take(sizeof(Control));     // contiguous from offset 0: zeroed by one memset
  L.off = take(sizeof(uint64_t) * 160); L.xs = take(kXsBytes); L.vox = take(4 * nvox);
  L.acc = take(with_acc ? 8 * nvox : 0);
  for (int p = 0; p < kMaxPipes; ++p) {
    Layout &Q = out[p]; Q = L;
    Q.ctl = ctl_at[p];
    Q.p0 = take(16 * batch); Q.p1 = take(16 * batch); Q.p2 = take(4 * batch);
    for (int k = 0; k < 3; ++k) Q.eq[k] = take((size_t)16 * L.eq_cap);
  }
  for (int p = 0; p < kMaxPipes; ++p) out[p].total = o;
}
static Layout make_layout(uint64_t batch, size_t nvox, bool with_acc) {
  Layout Ls[kMaxPipes]; make_layouts(batch, nvox, with_acc, Ls); return Ls[0];
}

int upload_tables(psl *P) {
  CUDA_TRY(cudaGetDevice(&P->device));
  const size_t G = P->groups.size();
  std::vector<uint32_t> let_off(G), n_let(G);
  std::vector<AliasEntry> table;
  for (size_t g = 0; g < G; ++g) {
    const HostGroup &hg = P->groups[g];
    let_off[g] = (uint32_t)table.size(); n_let[g] = (uint32_t)hg.ring.size();
    for (size_t i = 0; i < hg.ring.size(); ++i) {
      AliasEntry e; e.thresh = hg.thresh[i]; e.ring_c = hg.ring[i]; e.sector_c = hg.sector[i];
      e.ring_a = hg.ring[hg.alias[i]]; e.sector_a = hg.sector[hg.alias[i]]; e.pad = 0;
      table.push_back(e);
    }
  }
  P->total_lets = table.size();
  CUDA_TRY(cudaMalloc(&P->d_table, sizeof(AliasEntry) * std::max<size_t>(1, table.size())));
  CUDA_TRY(cudaMalloc((void **)&P->d_let_off, sizeof(uint32_t) * G));
  CUDA_TRY(cudaMalloc((void **)&P->d_n_let, sizeof(uint32_t) * G));
  CUDA_TRY(cudaMemcpy(P->d_table, table.data(), sizeof(AliasEntry) * table.size(), cudaMemcpyHostToDevice));
  CUDA_TRY(cudaMemcpy(P->d_let_off, let_off.data(), sizeof(uint32_t) * G, cudaMemcpyHostToDevice));
  CUDA_TRY(cudaMemcpy(P->d_n_let, n_let.data(), sizeof(uint32_t) * G, cudaMemcpyHostToDevice));
  // sigma_KN nodes for this model's energy range (the phantom-dependent majorant head is computed per launch)
  const double e_max = P->psr.e_min + P->psr.e_bin_width * P->n_ebin;
  P->xs_x0 = std::log2(0.045); P->xs_h = (std::log2(std::max(e_max, 0.1) * 1.001) - P->xs_x0) / kXsIntervals;
  CUDA_TRY(cudaMalloc(&P->d_xs, kXsBytes));
  k_build_xs<<<(kXsIntervals + 256) / 256, 256>>>(nullptr, (float *)P->d_xs, P->xs_x0, P->xs_h, kXsIntervals);
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaDeviceSynchronize());
  return MC_OK;
}

static void round_keys(uint64_t seed, uint32_t ks[20]) {
  for (int r = 0; r < 10; ++r) { ks[2 * r] = (uint32_t)seed + (uint32_t)r * 0x9E3779B9u; ks[2 * r + 1] = (uint32_t)(seed >> 32) + (uint32_t)r * 0xBB67AE85u; }
}

static SourceModel source_model(const psl &P) {
  SourceModel m{};
  m.table = (const AliasEntry *)P.d_table; m.let_off = P.d_let_off; m.n_let = P.d_n_let;
  m.n_groups = (int)P.groups.size(); m.n_ebin = P.n_ebin; m.n_sectors = P.n_sectors;
  m.e_min = (float)P.psr.e_min; m.e_bin_width = (float)P.psr.e_bin_width; m.ring_width = (float)P.psr.ring_width;
  m.z_phsp = (float)P.psr.z_phsp; m.inv_nsec = P.n_sectors > 0 ? (float)(1.0 / P.n_sectors) : 0.0f;
  m.let_mode = P.let_mode; m.grid_x0 = (float)P.grid_x0; m.let_size = (float)P.let_size;
  for (int s = 0; s < 3; ++s) { m.dir_tab[s] = (const float4 *)P.d_dir[s]; m.dir_K[s] = P.dir_K[s]; }
  m.n_ring = P.n_ring; m.jaw_dzx = (float)(P.jaws.z_jx - P.psr.z_phsp); m.jaw_dzy = (float)(P.jaws.z_jy - P.psr.z_phsp);
  const jaws_t &j = P.jaws;
  for (int s = 0; s < 3; ++s) {
    m.sigma_src[s] = (float)P.psr.sigma_src[s]; m.z_src[s] = (float)P.psr.z_src[s]; m.particle_type[s] = P.psr.particle_type[s];
    m.jaw_tx[s] = (float)((j.z_jx - P.psr.z_src[s]) / (P.psr.z_phsp - P.psr.z_src[s]));
    m.jaw_ty[s] = (float)((j.z_jy - P.psr.z_src[s]) / (P.psr.z_phsp - P.psr.z_src[s]));
  }
  m.jx_lo = (float)(j.x1 * j.z_jx / j.sad); m.jx_hi = (float)(j.x2 * j.z_jx / j.sad);
  m.jy_lo = (float)(j.y1 * j.z_jy / j.sad); m.jy_hi = (float)(j.y2 * j.z_jy / j.sad);
  return m;
}

static BeamXf beam_xf(const beam_geom_t &b) {
  BeamXf x{};
  for (int i = 0; i < 3; ++i) x.iso[i] = (float)b.iso[i];
  for (int i = 0; i < 9; ++i) x.R[i] = (float)b.R[i];
  x.sad = (float)b.sad;
  return x;
}

static Grid make_grid(const phantom_t &ph, long long *acc) {
  Grid g{};
  g.nx = ph.nx; g.ny = ph.ny; g.nz = ph.nz;
  g.ox = (float)ph.ox; g.oy = (float)ph.oy; g.oz = (float)ph.oz;
  g.dx = (float)ph.dx; g.dy = (float)ph.dy; g.dz = (float)ph.dz;
  g.idx = (float)(1.0 / ph.dx); g.idy = (float)(1.0 / ph.dy); g.idz = (float)(1.0 / ph.dz);
  g.density = ph.density; g.material = ph.material; g.acc = (unsigned long long *)acc;
  return g;
}

static bool phantom_ok(const phantom_t *ph) {
  return ph && ph->nx > 0 && ph->ny > 0 && ph->nz > 0 && ph->dx > 0 && ph->dy > 0 && ph->dz > 0 && ph->density && ph->material &&
         (uint64_t)ph->nx * ph->ny * ph->nz < 0x7fffffffull;
}

// Persistent-grid size: every SM filled to the kernel's occupancy.
// Fraction of the full persistent grid to launch.  When the packed phantom + int64 grid (12 B per voxel) do not fit L2,
// the kernels are bound by random DRAM sectors and fewer resident warps thrash less: measured on C4 (201 MB) 56.8 ms per
// 1e8 histories at 1.0, 53.1 at 0.75, 52.6 at 0.5; no effect on C1-C3 at 0.75, losses below (a single batch per pipeline
// then leaves SMs idle).
static double g_grid_scale = 1.0;

template <typename K>
static int persistent_blocks(K kernel, size_t smem = 0) {
  int dev = 0, sms = 0, per = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, kernel, kThreads, smem);
  return std::max(1, (int)(sms * std::max(1, per) * g_grid_scale));
}

// L2 residency for the packed phantom (north_star (4): "read-only 3D layout that is ... L2-resident").  The random
// voxel gathers of the transport kernels then hit L2 even when phantom + dose grid exceed it (C4: 64 MiB packed
// phantom + 128 MiB int64 grid against 126 MB of L2); everything else on the stream is marked streaming.
struct L2Window {
  cudaStream_t st = nullptr; bool on = false;
  void set(cudaStream_t s, const void *base, size_t bytes) {
    if (!getenv("PSLMC_L2_WINDOW")) return;       // opt-in: measured 11 % SLOWER on C4, neutral elsewhere
    int dev = 0; cudaGetDevice(&dev);
    int max_persist = 0, max_window = 0;
    cudaDeviceGetAttribute(&max_persist, cudaDevAttrMaxPersistingL2CacheSize, dev);
    cudaDeviceGetAttribute(&max_window, cudaDevAttrMaxAccessPolicyWindowSize, dev);
    if (max_persist <= 0 || max_window <= 0 || bytes < (8u << 20)) { cudaGetLastError(); return; }   // small phantoms stay in L2 anyway
    size_t cur = 0; cudaDeviceGetLimit(&cur, cudaLimitPersistingL2CacheSize);
    const size_t want = std::min<size_t>(bytes, (size_t)max_persist);
    if (cur < want && cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, want) != cudaSuccess) { cudaGetLastError(); return; }
    cudaStreamAttrValue v{};
    v.accessPolicyWindow.base_ptr = const_cast<void *>(base);
    v.accessPolicyWindow.num_bytes = std::min<size_t>(bytes, (size_t)max_window);
    v.accessPolicyWindow.hitRatio = (float)std::min(1.0, (double)want / (double)v.accessPolicyWindow.num_bytes);
    v.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
    v.accessPolicyWindow.missProp = cudaAccessPropertyNormal;
    if (cudaStreamSetAttribute(s, cudaStreamAttributeAccessPolicyWindow, &v) != cudaSuccess) { cudaGetLastError(); return; }
    st = s; on = true;
  }
  void clear() {
    if (!on) return;
    cudaStreamAttrValue v{};
    v.accessPolicyWindow.num_bytes = 0;
    cudaStreamSetAttribute(st, cudaStreamAttributeAccessPolicyWindow, &v);
    cudaCtxResetPersistingL2Cache();
    on = false;
  }
};

struct Timer {                                  // per-kernel-class CUDA-event timing (MC_FLAG_TIMING)
  bool on = false; cudaStream_t st = nullptr;
  std::vector<cudaEvent_t> ev[5];
  void begin(int cls) { if (!on) return; cudaEvent_t e; cudaEventCreate(&e); cudaEventRecord(e, st); ev[cls].push_back(e); }
  void end(int cls) { begin(cls); }
  void collect(float ms[5]) {
    for (int c = 0; c < 5; ++c) {
      ms[c] = 0;
      for (size_t i = 0; i + 1 < ev[c].size(); i += 2) { float t = 0; cudaEventElapsedTime(&t, ev[c][i], ev[c][i + 1]); ms[c] += t; }
      for (cudaEvent_t e : ev[c]) cudaEventDestroy(e);
      ev[c].clear();
    }
  }
};

// Everything the launch helpers need.
struct Run {
  cudaStream_t st; char *ws; Layout L; Grid g; Control *ctl;
  uint64_t seed, n_total, perm_a; int flags; bool dbg;
  unsigned long long *fp; uint64_t fp_base;
  Timer tm; uint64_t launches[5] = {0, 0, 0, 0, 0};
  int blocks_photon[2], blocks_electron[2];

  Queue queue(const size_t off[3], unsigned *count, unsigned cap) const {
    Queue q; q.a = (float4 *)(ws + off[0]); q.b = (float4 *)(ws + off[1]); q.c = (uint4 *)(ws + off[2]); q.count = count; q.cap = cap;
    return q;
  }
  TransportArgs base_args() const {
    TransportArgs a{};
    a.g = g; a.ctl = ctl; a.seed = seed; a.n_total = n_total; a.perm_a = perm_a;
    round_keys(seed, a.ks);
    a.p0 = (const float4 *)(ws + L.p0); a.p1 = (const float4 *)(ws + L.p1); a.p2 = g.com_index ? (const uint32_t *)(ws + L.p2) : nullptr;
    a.eq = queue(L.eq, &ctl->n_eq, L.eq_cap);
    a.fp = fp; a.fp_base = fp_base;
    a.electrons_local = (flags & MC_FLAG_ELECTRONS_LOCAL) ? 1 : 0;
    a.static_lanes = (flags & MC_FLAG_STATIC_LANES) ? 1 : 0;
    a.stage_scoring = (flags & MC_FLAG_STAGE_SCORING) ? 1 : 0;
    a.xs = xs; a.rhomax = rhomax ? rhomax : ctl->rhomax;
    return a;
  }
  XsTable xs{};
  const float *rhomax = nullptr;                 // where k_pack_phantom left the largest densities (pipeline 0's control block)
  static constexpr size_t kXsSmem = kXsBytes + sizeof(StageRing) * (kThreads / 32) + kAnnihBytes;   // k_photon dynamic shared memory
  // Builds the cross-section table of this call (after k_rhomax) for photon energies up to e_max.
  void build_xs(double e_max) {
    const double x0 = std::log2(0.045), x1 = std::log2(e_max * 1.001), hh = (x1 - x0) / kXsIntervals;
    float *nodes = (float *)(ws + L.xs);
    k_build_xs<<<(kXsIntervals + 256) / 256, 256, 0, st>>>(ctl, nodes, x0, hh, kXsIntervals);
    xs.data = nodes; xs.x0 = (float)x0; xs.inv_h = (float)(1.0 / hh); xs.n = kXsIntervals;
  }
  bool started = false;                         // a batch has been launched on this pipeline
  uint64_t batch = 0;                           // upper bound of the entries a photon launch can see
  int photon_blocks(int persistent) const { return (int)std::max<uint64_t>(1, std::min<uint64_t>({(uint64_t)persistent, (batch + kThreads - 1) / kThreads, 4096 / (kThreads / 32)})); }
  void photon(const TransportArgs &a) {
    tm.begin(MC_K_PHOTON);
    const int nb = photon_blocks(blocks_photon[dbg]);
    if (a.stage_scoring) {
      if (dbg) k_photon<true, true><<<nb, kThreads, kXsSmem + kScoreBytes, st>>>(a); else k_photon<false, true><<<nb, kThreads, kXsSmem + kScoreBytes, st>>>(a);
    } else {
      if (dbg) k_photon<true, false><<<nb, kThreads, kXsSmem, st>>>(a); else k_photon<false, false><<<nb, kThreads, kXsSmem, st>>>(a);
    }
    tm.end(MC_K_PHOTON); ++launches[MC_K_PHOTON];
  }
  void electron(const TransportArgs &a) {
    tm.begin(MC_K_ELECTRON);
    const int nb = blocks_electron[dbg];
    if (a.stage_scoring) {
      if (dbg) k_electron<true, true><<<nb, kThreads, kScoreBytes, st>>>(a); else k_electron<false, true><<<nb, kThreads, kScoreBytes, st>>>(a);
    } else {
      if (dbg) k_electron<true, false><<<nb, kThreads, 0, st>>>(a); else k_electron<false, false><<<nb, kThreads, 0, st>>>(a);
    }
    tm.end(MC_K_ELECTRON); ++launches[MC_K_ELECTRON];
  }
  void init_blocks() {
    const bool stage = (flags & MC_FLAG_STAGE_SCORING) != 0;
    if (stage) {
      cudaFuncSetAttribute(k_photon<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kXsSmem + kScoreBytes));
      cudaFuncSetAttribute(k_photon<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kXsSmem + kScoreBytes));
      blocks_photon[0] = persistent_blocks(k_photon<false, true>, kXsSmem + kScoreBytes); blocks_photon[1] = persistent_blocks(k_photon<true, true>, kXsSmem + kScoreBytes);
      blocks_electron[0] = persistent_blocks(k_electron<false, true>, kScoreBytes); blocks_electron[1] = persistent_blocks(k_electron<true, true>, kScoreBytes);
    } else {
      cudaFuncSetAttribute(k_photon<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kXsSmem);
      cudaFuncSetAttribute(k_photon<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kXsSmem);
      blocks_photon[0] = persistent_blocks(k_photon<false, false>, kXsSmem); blocks_photon[1] = persistent_blocks(k_photon<true, false>, kXsSmem);
      blocks_electron[0] = persistent_blocks(k_electron<false, false>); blocks_electron[1] = persistent_blocks(k_electron<true, false>);
    }
  }
  // Folds the finished batch's counters into the per-call totals and resets them.
  void next_batch() {
    tm.begin(MC_K_AUX); k_next_batch<<<1, 1, 0, st>>>(ctl); tm.end(MC_K_AUX); ++launches[MC_K_AUX];
  }
  const float4 *dbg_p0 = nullptr, *dbg_p1 = nullptr;
  // mc_transport_debug: photons of the caller's buffer, then every queued electron
  void transport_photon_debug(uint64_t first, const unsigned *count_ptr) {
    TransportArgs a = base_args();
    a.src_kind = SRC_BUFFER; a.buffer_is_debug = 1; a.first = first; a.want_type = 0;
    a.src_count = count_ptr; a.src_head = &ctl->head_pb; a.p0 = dbg_p0; a.p1 = dbg_p1;
    photon(a);
    drain_electrons();
  }
  // mc_dose: call right after k_sample.  The photons of the particle buffer (annihilation photons are transported
  // inside the launch by the converting lane), then every electron they queued.
  void transport_photon_batch(uint64_t first) {
    TransportArgs a = base_args();
    a.src_kind = SRC_BUFFER; a.buffer_is_debug = 0; a.first = first; a.want_type = 0;
    a.src_count = &ctl->n_pb; a.src_head = &ctl->head_pb;
    photon(a);
    drain_electrons();
  }
  void drain_electrons() {
    TransportArgs c = base_args();
    c.src_kind = SRC_QUEUE; c.src = c.eq; c.src_count = &ctl->n_eq; c.src_head = &ctl->head_eq;
    electron(c);
  }
  void transport_electron_buffer(uint64_t first, bool debug_buffer, const unsigned *count_ptr, unsigned *head) {
    TransportArgs a = base_args();
    a.src_kind = SRC_BUFFER; a.buffer_is_debug = debug_buffer; a.first = first; a.want_type = 1;
    a.src_count = count_ptr; a.src_head = head;
    electron(a);
  }
};

// Adds the per-call part of `src` (ledgers, counters, totals) into `dst` (pipelines are folded on the host).
static void merge_control(Control &dst, const Control &src) {
  for (int sl = 0; sl < kLedgerSlots; ++sl)
    for (int k = 0; k < 4; ++k) {
      unsigned __int128 a = ((unsigned __int128)dst.ledger[sl][k][1] << 64) | dst.ledger[sl][k][0];
      a += ((unsigned __int128)src.ledger[sl][k][1] << 64) | src.ledger[sl][k][0];
      dst.ledger[sl][k][0] = (unsigned long long)a; dst.ledger[sl][k][1] = (unsigned long long)(a >> 64);
    }
  for (int k = 0; k < ST_COUNT; ++k) dst.stat[k] += src.stat[k];
  dst.hw_eq = std::max(dst.hw_eq, src.hw_eq);
  dst.n_accepted += src.n_accepted; dst.n_missed += src.n_missed; dst.overflow |= src.overflow;
}

static void fold_stats(const Control &c, const Run &r, mc_stats_t *s) {
  for (int k = 0; k < 4; ++k) {
    unsigned __int128 tot = 0;
    for (int sl = 0; sl < kLedgerSlots; ++sl) tot += ((unsigned __int128)c.ledger[sl][k][1] << 64) | c.ledger[sl][k][0];
    s->ledger_hi[k] = (int64_t)(uint64_t)(tot >> 64); s->ledger_lo[k] = (uint64_t)tot;
  }
  s->n_missed = c.stat[ST_MISSED]; s->n_flights = c.stat[ST_FLIGHTS]; s->n_virtual = c.stat[ST_VIRTUAL];
  s->n_compton = c.stat[ST_COMPTON]; s->n_photo = c.stat[ST_PHOTO]; s->n_pair = c.stat[ST_PAIR];
  s->n_photon_cutoff = c.stat[ST_PCUT]; s->n_photon_escape = c.stat[ST_PESC]; s->n_uncollided_escape = c.stat[ST_UNCOLLIDED];
  s->n_sec_electrons = c.stat[ST_SEC_E]; s->n_sec_photons = c.stat[ST_SEC_P];
  s->n_electron_tracks = c.stat[ST_ETRACKS]; s->n_electron_steps = c.stat[ST_ESTEPS]; s->n_electron_escape = c.stat[ST_EESC];
  s->n_deposits = c.stat[ST_DEPOSITS];
  s->queue_high_water[0] = c.hw_eq; s->queue_high_water[1] = 0;    // no photon queue: annihilation photons stay in their lane
  for (int k = 0; k < 5; ++k) s->launches[k] = r.launches[k];
}

}  // namespace pslmc

using namespace pslmc;

static uint64_t gcd_u64(uint64_t a, uint64_t b) { while (b) { uint64_t t = a % b; a = b; b = t; } return a; }

// Mixed order (ablation): thread t handles history (a*t) mod N, a = smallest integer >= floor(0.618...N) coprime to N.
static uint64_t mixed_multiplier(uint64_t N) {
  if (N < 3) return 1;
  uint64_t a = (uint64_t)(0.6180339887 * (double)N);
  if (a < 1) a = 1;
  while (gcd_u64(a, N) != 1) ++a;
  return a;
}

// Number of pipelines of a call (PSLMC_PIPELINES = 1 switches the overlap off) and their streams (created once).
static int pipe_count(int requested) {
  const char *e = getenv("PSLMC_PIPELINES");
  const int n = requested > 0 ? requested : (e ? atoi(e) : kMaxPipes);
  return std::max(1, std::min(n, kMaxPipes));
}
static const std::vector<cudaStream_t> *pipe_streams() {
  static std::vector<cudaStream_t> st;
  static int dev_of = -1;
  int dev = 0; cudaGetDevice(&dev);
  if (st.empty() || dev_of != dev) {
    st.clear();
    for (int p = 0; p < kMaxPipes; ++p) {
      cudaStream_t s = nullptr;
      if (cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); st.clear(); return nullptr; }
      st.push_back(s);
    }
    dev_of = dev;
  }
  return &st;
}

// The driver proper.  All pointers inside `ph` are DEVICE pointers here.
static int run_dose(const psl_t *P, const phantom_t *ph, const beam_geom_t *beam, uint64_t N, uint64_t seed, uint64_t batch,
                    double *dose_out, const mc_opts_t *opts) {
  static const mc_opts_t kDefaults = {};
  if (!opts) opts = &kDefaults;
  if (!P || !beam || !phantom_ok(ph) || N == 0 || batch == 0 || batch > (1ull << 30) || (!dose_out && !opts->dose_acc))
    return fail(MC_E_INVALID_ARG, "mc_dose: invalid argument");
  const uint64_t hb = opts->history_begin, he = opts->history_end ? opts->history_end : N;
  if (hb > he || he > N) return fail(MC_E_INVALID_ARG, "mc_dose: history range outside [0, n_histories]");
  const bool mixed = opts->order == MC_ORDER_MIXED;
  if (mixed && (N >> 32)) return fail(MC_E_INVALID_ARG, "mc_dose: mixed order needs n_histories < 2^32");
  if (mixed && opts->fingerprints && (hb != 0 || he != N)) return fail(MC_E_INVALID_ARG, "mc_dose: mixed order + fingerprints needs the full range");
  if (opts->com_index && (!opts->com_dose || opts->com_rows < 1 || opts->com_cols != 2 * P->n_ebin * P->n_ring + P->n_ebin))
    return fail(MC_E_INVALID_ARG, "mc_dose: commissioning tally needs com_dose, com_rows >= 1 and com_cols = 2*n_ebin*n_ring + n_ebin");
  if (opts->com_index && mixed) return fail(MC_E_INVALID_ARG, "mc_dose: the commissioning tally runs in sorted order");
  int dev = 0; CUDA_TRY(cudaGetDevice(&dev));
  if (dev != P->device) return fail(MC_E_INVALID_ARG, "mc_dose: psl_t was built on another device");

  const size_t nvox = (size_t)ph->nx * ph->ny * ph->nz;
  Layout Ls[kMaxPipes];
  make_layouts(batch, nvox, opts->dose_acc == nullptr, Ls);
  const Layout &L = Ls[0];
  void *ws = opts->workspace;
  if (ws) { if (opts->workspace_bytes < L.total) return fail(MC_E_WORKSPACE, "mc_dose: workspace too small (see mc_workspace_bytes)"); }
  else { int rc = scratch_get(g_scratch, L.total, &ws); if (rc) return rc; }

  // Pipelines: batches are dealt round-robin to npipe independent launch sequences, each with its own control
  // block, particle buffer, queues and stream, all scoring into the one int64 grid.  Every transport kernel is
  // a persistent grid that fills the GPU, so the CTAs of one pipeline's next kernel start as the other
  // pipeline's kernel drains: the tails (lanes finishing their last, longest histories) overlap with useful
  // work instead of leaving SMs idle.  Integer tallies keep the result bit-identical for any npipe.
  const std::vector<cudaStream_t> *pstreams = nullptr;
  int npipe = pipe_count(opts->pipelines);
  if (npipe > 1 && !(pstreams = pipe_streams())) npipe = 1;
  cudaStream_t us = (cudaStream_t)opts->cuda_stream;
  long long *acc = opts->dose_acc ? (long long *)opts->dose_acc : (long long *)((char *)ws + L.acc);

  Run pipes[kMaxPipes];
  for (int p = 0; p < npipe; ++p) {
    Run &r = pipes[p];
    r.st = npipe > 1 ? (*pstreams)[p] : us; r.ws = (char *)ws; r.L = Ls[p]; r.ctl = (Control *)(r.ws + Ls[p].ctl);
    r.g = make_grid(*ph, acc); r.g.vox = (const uint32_t *)(r.ws + L.vox);
    r.g.com_index = (const int *)opts->com_index; r.g.com_dose = (unsigned long long *)opts->com_dose; r.g.com_rows = opts->com_rows;
    r.seed = seed; r.n_total = N; r.perm_a = mixed ? mixed_multiplier(N) : 0; r.flags = opts->flags; r.batch = batch;
    r.fp = (unsigned long long *)opts->fingerprints; r.fp_base = hb;
    r.dbg = (opts->flags & MC_FLAG_STATS) || opts->fingerprints || opts->com_index;   // the tally lives in the stats variants
    r.tm.on = (opts->flags & MC_FLAG_TIMING) != 0; r.tm.st = r.st;
    if (p == 0) { g_grid_scale = 12.0 * (double)nvox > 110e6 ? 0.75 : 1.0; r.init_blocks(); }
    else { for (int k = 0; k < 2; ++k) { r.blocks_photon[k] = pipes[0].blocks_photon[k]; r.blocks_electron[k] = pipes[0].blocks_electron[k]; } }
  }
  Run &r0 = pipes[0];

  std::vector<uint64_t> off(P->groups.size() + 1);
  allocate_host(*P, N, off.data());
  unsigned long long *d_off = (unsigned long long *)((char *)ws + L.off);

  // ---- prologue on the caller's stream
  cudaEvent_t ev0, ev1;
  CUDA_TRY(cudaEventCreate(&ev0)); CUDA_TRY(cudaEventCreate(&ev1));
  CUDA_TRY(cudaEventRecord(ev0, us));
  CUDA_TRY(cudaMemsetAsync(ws, 0, align_up(sizeof(Control)) * kMaxPipes, us));          // every pipeline's control block
  CUDA_TRY(cudaMemcpyAsync(d_off, off.data(), sizeof(uint64_t) * off.size(), cudaMemcpyHostToDevice, us));
  if (!opts->dose_acc) CUDA_TRY(cudaMemsetAsync(acc, 0, 8 * nvox, us));
  Timer tm_us; tm_us.on = r0.tm.on; tm_us.st = us;
  uint64_t launches_us[5] = {0, 0, 0, 0, 0};
  tm_us.begin(MC_K_AUX);
  k_pack_phantom<<<592, 256, 0, us>>>(ph->density, ph->material, nvox, (uint32_t *)((char *)ws + L.vox), r0.ctl);
  r0.xs.data = (const float *)P->d_xs; r0.xs.x0 = (float)P->xs_x0; r0.xs.inv_h = (float)(1.0 / P->xs_h); r0.xs.n = kXsIntervals;
  tm_us.end(MC_K_AUX); launches_us[MC_K_AUX] += 1;
  for (int p = 0; p < npipe; ++p) { pipes[p].xs = r0.xs; pipes[p].rhomax = r0.ctl->rhomax; }
  L2Window l2w; l2w.set(us, (char *)ws + L.vox, 4 * nvox);
  cudaEvent_t ev_fork = nullptr, ev_join[kMaxPipes] = {};
  if (npipe > 1) {
    CUDA_TRY(cudaEventCreateWithFlags(&ev_fork, cudaEventDisableTiming));
    CUDA_TRY(cudaEventRecord(ev_fork, us));
    for (int p = 0; p < npipe; ++p) CUDA_TRY(cudaStreamWaitEvent(pipes[p].st, ev_fork, 0));
  }

  SampleArgs sa[kMaxPipes];
  for (int p = 0; p < npipe; ++p) {
    Run &r = pipes[p]; SampleArgs &a = sa[p]; a = SampleArgs{};
    a.m = source_model(*P); a.beam = beam_xf(*beam); a.off_g = d_off; a.seed = seed; round_keys(seed, a.ks); a.n_total = N; a.perm_a = r.perm_a;
    a.p0 = (float4 *)(r.ws + r.L.p0); a.p1 = (float4 *)(r.ws + r.L.p1); a.ctl = r.ctl; a.fp = r.fp; a.fp_base = hb; a.compact = 1; a.g = r.g; a.stats = r.dbg ? 1 : 0;
    a.p2 = r.g.com_index ? (uint32_t *)(r.ws + r.L.p2) : nullptr;
  }

  memset(&g_stats, 0, sizeof g_stats);
  auto sample_batch = [&](int p, uint64_t first, uint64_t count) {
    Run &r = pipes[p];
    if (r.started) r.next_batch();                      // (a pipeline's first batch finds the control block freshly zeroed)
    r.started = true;
    sa[p].first = first; sa[p].count = (unsigned)count;
    r.tm.begin(MC_K_SAMPLE);
    k_sample<<<(unsigned)((count + kThreads - 1) / kThreads), kThreads, 0, r.st>>>(sa[p]);
    r.tm.end(MC_K_SAMPLE); ++r.launches[MC_K_SAMPLE];
  };
  const int ne = P->n_ebin;
  uint64_t task = 0;
  if (!mixed) {
    // one sub-source type at a time, energy bins ascending, M histories per launch
    for (int s = 0; s < 3; ++s) {
      const uint64_t lo = std::max(hb, off[(size_t)s * ne]), hi = std::min(he, off[(size_t)(s + 1) * ne]);
      if (lo >= hi) continue;
      g_stats.n_hist[s] = hi - lo;
      // equal batches: ceil(n / batch) launches of the same size (a short last batch is mostly tail)
      const uint64_t nb = (hi - lo + batch - 1) / batch, even = std::min(batch, (((hi - lo + nb - 1) / nb) + kThreads - 1) / kThreads * kThreads);
      for (uint64_t first = lo; first < hi; first += even, ++task) {
        const int p = (int)(task % npipe); Run &r = pipes[p];
        sample_batch(p, first, std::min(even, hi - first));
        if (P->psr.particle_type[s] == 0) r.transport_photon_batch(first);
        else r.transport_electron_buffer(first, false, &r.ctl->n_pb, &r.ctl->head_pb);
      }
    }
  } else {
    for (int s = 0; s < 3; ++s) g_stats.n_hist[s] = 0;     // mixed: per-type counts are not tracked per range
    for (uint64_t first = hb; first < he; first += batch, ++task) {
      const int p = (int)(task % npipe); Run &r = pipes[p];
      sample_batch(p, first, std::min(batch, he - first));
      r.transport_electron_buffer(first, false, &r.ctl->n_pb, &r.ctl->pad0);
      r.transport_photon_batch(first);
    }
    if (hb == 0 && he == N) for (int s = 0; s < 3; ++s) g_stats.n_hist[s] = off[(size_t)(s + 1) * ne] - off[(size_t)s * ne];
  }
  for (int p = 0; p < npipe; ++p) {
    Run &r = pipes[p];                                // (the last batch's counters are folded on the host, below: no launch)
    if (npipe > 1) {
      CUDA_TRY(cudaEventCreateWithFlags(&ev_join[p], cudaEventDisableTiming));
      CUDA_TRY(cudaEventRecord(ev_join[p], r.st));
      CUDA_TRY(cudaStreamWaitEvent(us, ev_join[p], 0));
    }
  }
  if (dose_out) {
    tm_us.begin(MC_K_FINALISE);
    const double inv_vn = 1.0 / (ph->dx * ph->dy * ph->dz * (double)N);
    k_finalise<<<592, 256, 0, us>>>(acc, ph->density, nvox, inv_vn, dose_out);
    tm_us.end(MC_K_FINALISE); ++launches_us[MC_K_FINALISE];
  }
  CUDA_TRY(cudaEventRecord(ev1, us));
  CUDA_TRY(cudaGetLastError());
  Control hc[kMaxPipes];
  for (int p = 0; p < npipe; ++p) CUDA_TRY(cudaMemcpyAsync(&hc[p], pipes[p].ctl, sizeof(Control), cudaMemcpyDeviceToHost, us));
  CUDA_TRY(cudaStreamSynchronize(us));
  for (int p = 0; p < npipe; ++p) {                     // what k_next_batch would have folded for the last batch of each pipeline
    hc[p].n_accepted += hc[p].n_pb; hc[p].hw_eq = std::max(hc[p].hw_eq, hc[p].n_eq);
  }
  l2w.clear();
  CUDA_TRY(cudaEventElapsedTime(&g_stats.ms_total, ev0, ev1));
  cudaEventDestroy(ev0); cudaEventDestroy(ev1);
  if (ev_fork) cudaEventDestroy(ev_fork);
  for (int p = 0; p < npipe; ++p) if (ev_join[p]) cudaEventDestroy(ev_join[p]);
  // fold the pipelines: kernel-class times add up (they overlap in wall time), counters and ledgers sum exactly
  tm_us.collect(g_stats.ms);
  for (int p = 0; p < npipe; ++p) {
    float ms[5]; pipes[p].tm.collect(ms);
    for (int k = 0; k < 5; ++k) { g_stats.ms[k] += ms[k]; launches_us[k] += pipes[p].launches[k]; }
    if (p > 0) merge_control(hc[0], hc[p]);
  }
  for (int k = 0; k < 5; ++k) r0.launches[k] = launches_us[k];
  fold_stats(hc[0], r0, &g_stats);
  g_stats.n_jaw_rejected = (he - hb) - hc[0].n_accepted - hc[0].n_missed;
  if (hc[0].overflow) return fail(MC_E_OVERFLOW, "mc_dose: a secondary queue overflowed; use a larger batch workspace");
  return MC_OK;
}

extern "C" void psl_free(psl_t *P) {
  if (!P) return;
  if (P->d_table) cudaFree(P->d_table);
  if (P->d_let_off) cudaFree(P->d_let_off);
  if (P->d_n_let) cudaFree(P->d_n_let);
  for (int s = 0; s < 3; ++s) if (P->d_dir[s]) cudaFree(P->d_dir[s]);
  if (P->d_xs) cudaFree(P->d_xs);
  delete P;
}

extern "C" int psl_set_direction_model(psl_t *P, int32_t stype, int32_t K, const double *c, const double *mu,
                                       const double *sigma_a, const double *sigma_b) {
  if (!P || stype < 0 || stype > 2 || K < 0 || K > 8 || (K > 0 && (!c || !mu || !sigma_a || !sigma_b)))
    return fail(MC_E_INVALID_ARG, "psl_set_direction_model: invalid argument");
  if (P->d_dir[stype]) { cudaFree(P->d_dir[stype]); P->d_dir[stype] = nullptr; }
  P->dir_K[stype] = 0;
  if (K == 0) return MC_OK;
  const size_t cells = (size_t)P->n_ebin * P->n_ring, n = cells * K;
  std::vector<float> tab(4 * n);
  for (size_t b = 0; b < n; b += K) {
    double tot = 0, run = 0;
    for (int k = 0; k < K; ++k) { if (!(c[b + k] >= 0) || !(sigma_a[b + k] >= 0) || !(sigma_b[b + k] >= 0)) return fail(MC_E_INVALID_ARG, "psl_set_direction_model: negative weight or sigma"); tot += c[b + k]; }
    if (!(tot > 0)) return fail(MC_E_INVALID_ARG, "psl_set_direction_model: a (bin, ring) cell has no weight");
    for (int k = 0; k < K; ++k) {
      run += c[b + k];
      float *o = &tab[4 * (b + k)];
      o[0] = (float)(run / tot); o[1] = (float)mu[b + k]; o[2] = (float)sigma_a[b + k]; o[3] = (float)sigma_b[b + k];
    }
  }
  CUDA_TRY(cudaMalloc(&P->d_dir[stype], sizeof(float) * tab.size()));
  CUDA_TRY(cudaMemcpy(P->d_dir[stype], tab.data(), sizeof(float) * tab.size(), cudaMemcpyHostToDevice));
  P->dir_K[stype] = K;
  return MC_OK;
}

extern "C" size_t mc_workspace_bytes(const psl_t *P, const phantom_t *ph, uint64_t batch) {
  if (!P || !ph || ph->nx <= 0 || ph->ny <= 0 || ph->nz <= 0 || batch == 0 || batch > (1ull << 30)) return 0;
  return make_layout(batch, (size_t)ph->nx * ph->ny * ph->nz, true).total;
}

extern "C" int mc_dose(const psl_t *P, const phantom_t *ph, const beam_geom_t *beam, uint64_t n_histories, uint64_t seed,
                       uint64_t batch, double *dose_out, const mc_opts_t *opts) {
  return run_dose(P, ph, beam, n_histories, seed, batch, dose_out, opts);
}

extern "C" int mc_dose_host(const psl_t *P, const phantom_t *ph, const beam_geom_t *beam, uint64_t n_histories, uint64_t seed,
                            uint64_t batch, double *dose_out_host, const mc_opts_t *opts) {
  if (!ph || ph->nx <= 0 || ph->ny <= 0 || ph->nz <= 0 || !ph->density || !ph->material || !dose_out_host)
    return fail(MC_E_INVALID_ARG, "mc_dose_host: invalid argument");
  const size_t nvox = (size_t)ph->nx * ph->ny * ph->nz;
  const size_t o_rho = 0, o_mat = align_up(4 * nvox), o_dose = o_mat + align_up(nvox), total = o_dose + 8 * nvox;
  void *io = nullptr;
  int rc = scratch_get(g_hostio, total, &io); if (rc) return rc;
  cudaStream_t st = opts ? (cudaStream_t)opts->cuda_stream : nullptr;
  char *b = (char *)io;
  CUDA_TRY(cudaMemcpyAsync(b + o_rho, ph->density, 4 * nvox, cudaMemcpyHostToDevice, st));
  CUDA_TRY(cudaMemcpyAsync(b + o_mat, ph->material, nvox, cudaMemcpyHostToDevice, st));
  phantom_t d = *ph; d.density = (const float *)(b + o_rho); d.material = (const uint8_t *)(b + o_mat);
  rc = run_dose(P, &d, beam, n_histories, seed, batch, (double *)(b + o_dose), opts);
  if (rc) return rc;
  CUDA_TRY(cudaMemcpyAsync(dose_out_host, b + o_dose, 8 * nvox, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  return MC_OK;
}

extern "C" int mc_stats(mc_stats_t *out) {
  if (!out) return fail(MC_E_INVALID_ARG, "mc_stats: null argument");
  *out = g_stats;
  return MC_OK;
}

// ---------------------------------------------------------------- parity / debug exports
extern "C" int mc_sample_debug(const psl_t *P, const beam_geom_t *beam, uint64_t first_history, uint64_t count,
                               uint64_t n_histories, uint64_t seed, float *soa_out, void *cuda_stream) {
  if (!P || !beam || n_histories == 0 || first_history + count > n_histories || count > 0x7fffffffull)
    return fail(MC_E_INVALID_ARG, "mc_sample_debug: invalid argument");
  if (count == 0) return MC_OK;
  if (!soa_out) return fail(MC_E_INVALID_ARG, "mc_sample_debug: soa_out is null");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  std::vector<uint64_t> off(P->groups.size() + 1);
  allocate_host(*P, n_histories, off.data());
  void *d_off = nullptr;
  CUDA_TRY(cudaMalloc(&d_off, sizeof(uint64_t) * off.size()));
  CUDA_TRY(cudaMemcpyAsync(d_off, off.data(), sizeof(uint64_t) * off.size(), cudaMemcpyHostToDevice, st));
  SampleArgs sa{};
  sa.m = source_model(*P); sa.beam = beam_xf(*beam); sa.off_g = (const unsigned long long *)d_off;
  sa.seed = seed; round_keys(seed, sa.ks); sa.first = first_history; sa.n_total = n_histories; sa.perm_a = 0; sa.count = (unsigned)count;
  sa.p0 = (float4 *)soa_out; sa.p1 = (float4 *)soa_out + count; sa.ctl = nullptr; sa.fp = nullptr; sa.compact = 0;
  k_sample<<<(unsigned)((count + kThreads - 1) / kThreads), kThreads, 0, st>>>(sa);
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaStreamSynchronize(st));
  cudaFree(d_off);
  return MC_OK;
}

extern "C" int mc_transport_debug(const phantom_t *ph, int32_t particle_type, const float *soa_in, uint64_t first_history,
                                  uint64_t count, uint64_t seed, const mc_opts_t *opts) {
  if (!phantom_ok(ph) || !soa_in || !opts || !opts->dose_acc || (particle_type != 0 && particle_type != 1) || count > (1ull << 30))
    return fail(MC_E_INVALID_ARG, "mc_transport_debug: invalid argument (opts->dose_acc is required)");
  memset(&g_stats, 0, sizeof g_stats);
  if (count == 0) return MC_OK;
  const size_t nvox = (size_t)ph->nx * ph->ny * ph->nz;
  const Layout L = make_layout(count, nvox, false);
  void *ws = opts->workspace;
  if (ws) { if (opts->workspace_bytes < L.total) return fail(MC_E_WORKSPACE, "mc_transport_debug: workspace too small"); }
  else { int rc = scratch_get(g_scratch, L.total, &ws); if (rc) return rc; }
  Run r{};
  r.st = (cudaStream_t)opts->cuda_stream; r.ws = (char *)ws; r.L = L; r.ctl = (Control *)(r.ws + L.ctl);
  r.g = make_grid(*ph, (long long *)opts->dose_acc); r.g.vox = (const uint32_t *)(r.ws + L.vox);
  r.seed = seed; r.n_total = first_history + count; r.perm_a = 0; r.flags = opts->flags; r.batch = count;
  r.fp = (unsigned long long *)opts->fingerprints; r.fp_base = first_history;
  r.dbg = true; r.tm.on = false; g_grid_scale = 1.0; r.init_blocks();
  cudaEvent_t ev0, ev1;
  CUDA_TRY(cudaEventCreate(&ev0)); CUDA_TRY(cudaEventCreate(&ev1));
  CUDA_TRY(cudaEventRecord(ev0, r.st));
  CUDA_TRY(cudaMemsetAsync(r.ctl, 0, sizeof(Control), r.st));
  k_pack_phantom<<<592, 256, 0, r.st>>>(ph->density, ph->material, nvox, (uint32_t *)(r.ws + r.L.vox), r.ctl);
  r.build_xs(64.0);                              // debug entry: energies up to 64 MeV
  // the caller's planes stand in for the particle buffer; n_pb = count
  const unsigned cnt = (unsigned)count;
  CUDA_TRY(cudaMemcpyAsync(&r.ctl->n_pb, &cnt, sizeof cnt, cudaMemcpyHostToDevice, r.st));
  TransportArgs a = r.base_args();
  a.p0 = (const float4 *)soa_in; a.p1 = (const float4 *)soa_in + count;
  a.src_kind = SRC_BUFFER; a.buffer_is_debug = 1; a.first = first_history; a.want_type = particle_type;
  a.src_count = &r.ctl->n_pb; a.src_head = &r.ctl->head_pb;
  if (particle_type == 0) {
    r.dbg_p0 = (const float4 *)soa_in; r.dbg_p1 = (const float4 *)soa_in + count;
    r.transport_photon_debug(first_history, &r.ctl->n_pb);
  } else {
    r.electron(a);
  }
  k_next_batch<<<1, 1, 0, r.st>>>(r.ctl);
  CUDA_TRY(cudaEventRecord(ev1, r.st));
  CUDA_TRY(cudaGetLastError());
  Control hc;
  CUDA_TRY(cudaMemcpyAsync(&hc, r.ctl, sizeof(Control), cudaMemcpyDeviceToHost, r.st));
  CUDA_TRY(cudaStreamSynchronize(r.st));
  CUDA_TRY(cudaEventElapsedTime(&g_stats.ms_total, ev0, ev1));
  cudaEventDestroy(ev0); cudaEventDestroy(ev1);
  fold_stats(hc, r, &g_stats);
  if (hc.overflow) return fail(MC_E_OVERFLOW, "mc_transport_debug: a secondary queue overflowed");
  return MC_OK;
}

extern "C" int mc_xs_debug(const float rhomax[3], double e_max, const float *E_host, uint64_t n, float *out_host) {
  if (!rhomax || !E_host || !out_host || !(e_max > 0.05) || n > (1ull << 28)) return fail(MC_E_INVALID_ARG, "mc_xs_debug: invalid argument");
  if (n == 0) return MC_OK;
  char *d = nullptr;
  const size_t o_ctl = 0, o_xs = align_up(sizeof(Control)), o_e = o_xs + align_up(kXsBytes), o_out = o_e + align_up(4 * n), total = o_out + 12 * n;
  CUDA_TRY(cudaMalloc((void **)&d, total));
  Control hc; memset(&hc, 0, sizeof hc);
  for (int k = 0; k < 3; ++k) hc.rhomax[k] = rhomax[k];
  CUDA_TRY(cudaMemcpy(d + o_ctl, &hc, sizeof hc, cudaMemcpyHostToDevice));
  CUDA_TRY(cudaMemcpy(d + o_e, E_host, 4 * n, cudaMemcpyHostToDevice));
  Run r{}; r.st = nullptr; r.ws = d; r.L.xs = o_xs; r.ctl = (Control *)(d + o_ctl);
  r.build_xs(e_max);
  k_xs_debug<<<(unsigned)((n + 255) / 256), 256>>>(r.xs, (const float *)(d + o_e), n, (float *)(d + o_out));
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaMemcpy(out_host, d + o_out, 12 * n, cudaMemcpyDeviceToHost));
  cudaFree(d);
  return MC_OK;
}

extern "C" int mc_atomic_peak_debug(int64_t *acc, uint64_t nvox, uint64_t n_ops, uint64_t seed, float *ms_out) {
  if (!acc || !ms_out || nvox == 0 || nvox >= 0x7fffffffull || n_ops == 0) return fail(MC_E_INVALID_ARG, "mc_atomic_peak_debug: invalid argument");
  int dev = 0, sms = 0; CUDA_TRY(cudaGetDevice(&dev));
  CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const unsigned blocks = (unsigned)sms * 8, threads = blocks * kThreads;
  const unsigned per_thread = (unsigned)std::max<uint64_t>(1, n_ops / threads);
  cudaEvent_t e0, e1; CUDA_TRY(cudaEventCreate(&e0)); CUDA_TRY(cudaEventCreate(&e1));
  k_atomic_peak<<<blocks, kThreads>>>((unsigned long long *)acc, (unsigned)nvox, 16u, (unsigned)seed);      // warm-up
  CUDA_TRY(cudaEventRecord(e0));
  k_atomic_peak<<<blocks, kThreads>>>((unsigned long long *)acc, (unsigned)nvox, per_thread, (unsigned)seed + 1u);
  CUDA_TRY(cudaEventRecord(e1));
  CUDA_TRY(cudaEventSynchronize(e1));
  CUDA_TRY(cudaEventElapsedTime(ms_out, e0, e1));
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  ms_out[1] = (float)((double)per_thread * threads);
  return MC_OK;
}

extern "C" int mc_philox_debug(uint64_t seed, uint64_t history, uint32_t track, uint32_t block, uint32_t *out) {
  if (!out) return fail(MC_E_INVALID_ARG, "mc_philox_debug: null argument");
  uint32_t *d = nullptr;
  CUDA_TRY(cudaMalloc((void **)&d, 16));
  k_philox_debug<<<1, 1>>>(seed, history, track, block, d);
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaMemcpy(out, d, 16, cudaMemcpyDeviceToHost));
  cudaFree(d);
  return MC_OK;
}
