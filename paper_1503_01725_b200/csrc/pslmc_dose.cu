// pslmc_dose.cu — the batching driver and the C ABI of the hot path: iterated k_sample → k_photon /
// k_electron launches per sub-source type and energy order, the electron
// queue, int64 scoring, finalise, stats.  No CPU fallback: every entry point here needs a device.
// No process-global device state: scratch and streams are the caller's (include/pslmc.h).
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

static size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

// Workspace layout for a batch of B primaries.  Shared by the whole call: control blocks, cross-section
// data, packed phantom, the int64 dose grid (used when the caller gives no dose_acc).  Per pipeline
// (kMaxPipes of them, see Session): the particle buffer (2 planes + the commissioning column) twice - as packed by
// k_sample and ordered by entry tile -, the entry-tile counters, and the electron queue (capacity 4B, 3 planes).  mc_dose_host appends its staging area (phantom in, dose out).
constexpr int kMaxPipes = 3;     // two on the caller's aux_streams, the third on cuda_stream itself
struct Layout {
  size_t ctl[kMaxPipes], tile[kMaxPipes], xs, vox, brick, sbrick, com_mask, com_coarse, acc, p0[kMaxPipes], p1[kMaxPipes], p2[kMaxPipes], q0[kMaxPipes], q1[kMaxPipes], q2[kMaxPipes],
      eq[kMaxPipes][3], total, zero_bytes;
  size_t host_rho, host_mat, host_dose, host_total;
  unsigned eq_cap;
};
static size_t brick_count(int nx, int ny, int nz) { return (size_t)((nx + 3) / 4) * ((ny + 3) / 4) * ((nz + 3) / 4); }
static Layout make_layout(uint64_t batch, size_t nvox, size_t nbricks) {
  Layout L{}; size_t o = 0;
  auto take = [&](size_t b) { size_t at = o; o += align_up(b); return at; };
  L.eq_cap = (unsigned)std::min<uint64_t>(4 * batch, 0x7fffffffu);
  for (int p = 0; p < kMaxPipes; ++p) L.ctl[p] = take(sizeof(Control));     // contiguous from offset 0: zeroed by one memset,
  for (int p = 0; p < kMaxPipes; ++p) L.tile[p] = take(2 * sizeof(unsigned) * kTileBinsMax);   // with the entry-tile counts and cursors
  L.com_coarse = take(4 * ((nvox >> 14) + 1));               // commissioning tally: one bit per 512 voxels (zeroed with the rest)
  L.zero_bytes = o;
  L.xs = take(kXsBytes); L.vox = take(4 * nvox); L.brick = take(4 * nbricks); L.sbrick = take(4 * nbricks);     // (super-bricks <= bricks for any grid shape)
  L.com_mask = take(4 * ((nvox + 31) / 32)); L.acc = take(8 * nvox);
  for (int p = 0; p < kMaxPipes; ++p) {
    L.p0[p] = take(16 * batch); L.p1[p] = take(16 * batch); L.p2[p] = take(4 * batch);
    L.q0[p] = take(16 * batch); L.q1[p] = take(16 * batch); L.q2[p] = take(4 * batch);     // the same, ordered by entry tile
    for (int k = 0; k < 3; ++k) L.eq[p][k] = take((size_t)16 * L.eq_cap);
  }
  L.total = o;
  L.host_rho = take(4 * nvox); L.host_mat = take(nvox); L.host_dose = take(8 * nvox);
  L.host_total = o;
  return L;
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

// Persistent-grid size: every SM filled to the kernel's occupancy, times `scale`.
template <typename K>
static int persistent_blocks(K kernel, size_t smem, double scale) {
  int dev = 0, sms = 0, per = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, kernel, kThreads, smem);
  return std::max(1, (int)(sms * std::max(1, per) * scale));
}

struct Timer {                                  // per-kernel-class CUDA-event timing (MC_FLAG_TIMING)
  bool on = false; cudaStream_t st = nullptr;
  std::vector<cudaEvent_t> ev[5];
  void begin(int cls) { if (!on) return; cudaEvent_t e; cudaEventCreate(&e); cudaEventRecord(e, st); ev[cls].push_back(e); }
  void end(int cls) { begin(cls); }
  void discard() { for (auto &v : ev) { for (cudaEvent_t e : v) cudaEventDestroy(e); v.clear(); } }
  void collect(float ms[5]) {
    for (int c = 0; c < 5; ++c) {
      ms[c] = 0;
      for (size_t i = 0; i + 1 < ev[c].size(); i += 2) { float t = 0; cudaEventElapsedTime(&t, ev[c][i], ev[c][i + 1]); ms[c] += t; }
      for (cudaEvent_t e : ev[c]) cudaEventDestroy(e);
      ev[c].clear();
    }
  }
};

// One launch sequence ("pipeline"): its stream, control block, particle buffer and electron queue.
struct Pipe {
  cudaStream_t st = nullptr; Control *ctl = nullptr;
  float4 *p0 = nullptr, *p1 = nullptr; uint32_t *p2 = nullptr;      // packed by k_sample
  float4 *q0 = nullptr, *q1 = nullptr; uint32_t *q2 = nullptr;      // ordered by entry tile (what the transport kernels read when tiles are on)
  unsigned *tile_count = nullptr, *tile_cursor = nullptr;
  Queue eq{};
  Timer tm; uint64_t launches[5] = {0, 0, 0, 0, 0};
  bool started = false;                         // a batch has been launched on this pipeline
};

// Everything one mc_dose / mc_plan_dose / mc_transport_debug call shares: workspace, phantom, kernel variants,
// pipelines.  begin() → any number of run_beam() → end().  Nothing in between returns to the host: kernels read
// their input counts from the device control blocks; end() synchronises once.
struct Session {
  char *ws = nullptr; Layout L{}; Grid g{}; size_t nvox = 0;
  cudaStream_t us = nullptr;                    // the caller's stream
  int npipe = 1; Pipe pipes[kMaxPipes];
  int flags = 0, mode = MODE_PLAIN; bool dbg = false, timing = false;
  unsigned eq_cap = 0; uint64_t batch = 0;
  XsTable xs{}; const float *rhomax = nullptr;
  int blocks_photon = 1, blocks_electron = 1, blocks_sample = 1, sms = 1;
  TileMap tm{};                                 // nbins = 0: batches are not ordered by entry tile
  uint64_t task = 0;                            // batches dealt so far (round-robin over the pipelines)
  cudaEvent_t ev0 = nullptr, ev1 = nullptr, ev_fork = nullptr, ev_join[kMaxPipes] = {};
  Timer tm_us; uint64_t launches_us[5] = {0, 0, 0, 0, 0};
  unsigned long long *fp = nullptr; uint64_t fp_base = 0;
  static constexpr size_t kXsSmem = kXsBytes + sizeof(StageRing) * (kThreads / 32) + kAnnihBytes;   // k_photon dynamic shared memory

  ~Session() {
    for (cudaEvent_t e : {ev0, ev1, ev_fork, ev_join[0], ev_join[1], ev_join[2]}) if (e) cudaEventDestroy(e);
    tm_us.discard(); for (Pipe &p : pipes) p.tm.discard();                      // (events left by an early error return)
  }

  // Kernel variants: <stats + fingerprints + commissioning tally> or plain, <shared-memory staging of the scoring> or not.
  // Kernel variants: mode (plain / + commissioning tally / + stats and fingerprints) x shared-memory staging of the scoring.
  template <int M, bool S> void launch_photon_v(Pipe &p, const TransportArgs &a, int nb, size_t sm) { k_photon<M, S><<<nb, kThreads, sm, p.st>>>(a); }
  template <int M, bool S> void launch_electron_v(Pipe &p, const TransportArgs &a, int nb, size_t sm) { k_electron<M, S><<<nb, kThreads, sm, p.st>>>(a); }
#define PSLMC_DISPATCH(fn, ...)                                                                                     \
  do {                                                                                                              \
    const bool st_ = (flags & MC_FLAG_STAGE_SCORING) != 0;                                                          \
    if (mode == MODE_PLAIN) { if (st_) fn<MODE_PLAIN, true>(__VA_ARGS__); else fn<MODE_PLAIN, false>(__VA_ARGS__); } \
    else if (mode == MODE_COM) { if (st_) fn<MODE_COM, true>(__VA_ARGS__); else fn<MODE_COM, false>(__VA_ARGS__); }  \
    else { if (st_) fn<MODE_DBG, true>(__VA_ARGS__); else fn<MODE_DBG, false>(__VA_ARGS__); }                        \
  } while (0)
  void launch_photon(Pipe &p, const TransportArgs &a) {
    p.tm.begin(MC_K_PHOTON);
    const int nb = (int)std::max<uint64_t>(1, std::min<uint64_t>({(uint64_t)blocks_photon, (batch + kThreads - 1) / kThreads, 4096 / (kThreads / 32)}));
    const size_t sm = kXsSmem + (a.stage_scoring ? kScoreBytes : 0);
    PSLMC_DISPATCH(launch_photon_v, p, a, nb, sm);
    p.tm.end(MC_K_PHOTON); ++p.launches[MC_K_PHOTON];
  }
  void launch_electron(Pipe &p, const TransportArgs &a) {
    p.tm.begin(MC_K_ELECTRON);
    const int nb = blocks_electron; const size_t sm = a.stage_scoring ? kScoreBytes : 0;
    PSLMC_DISPATCH(launch_electron_v, p, a, nb, sm);
    p.tm.end(MC_K_ELECTRON); ++p.launches[MC_K_ELECTRON];
  }
  template <int M, bool S> void setup_v(size_t smp, size_t sme, double scale) {
    cudaFuncSetAttribute(k_photon<M, S>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smp);
    blocks_photon = persistent_blocks(k_photon<M, S>, smp, scale);
    blocks_electron = persistent_blocks(k_electron<M, S>, sme, scale);
  }
  void init_blocks(double scale) {
    const bool stage = (flags & MC_FLAG_STAGE_SCORING) != 0;
    const size_t smp = kXsSmem + (stage ? kScoreBytes : 0), sme = stage ? kScoreBytes : 0;
    PSLMC_DISPATCH(setup_v, smp, sme, scale);
  }
#undef PSLMC_DISPATCH

  TransportArgs base_args(const Pipe &p, uint64_t seed, uint64_t n_total, uint64_t perm_a) const {
    TransportArgs a{};
    a.g = g; a.ctl = p.ctl; a.seed = seed; a.n_total = n_total; a.perm_a = perm_a;
    round_keys(seed, a.ks);
    const bool tiles = tm.nbins > 0;
    a.p0 = tiles ? p.q0 : p.p0; a.p1 = tiles ? p.q1 : p.p1; a.p2 = g.com_index ? (tiles ? p.q2 : p.p2) : nullptr;
    a.eq = p.eq;
    a.fp = fp; a.fp_base = fp_base;
    a.electrons_local = (flags & MC_FLAG_ELECTRONS_LOCAL) ? 1 : 0;
    a.static_lanes = (flags & MC_FLAG_STATIC_LANES) ? 1 : 0;
    a.stage_scoring = (flags & MC_FLAG_STAGE_SCORING) ? 1 : 0;
    a.fp_voxels = (flags & MC_FLAG_FP_VOXELS) ? 1 : 0;
    a.xs = xs; a.rhomax = rhomax;
    return a;
  }
  void drain_electrons(Pipe &p, const TransportArgs &base) {
    TransportArgs c = base;
    c.src_kind = SRC_QUEUE; c.src = c.eq; c.src_count = &p.ctl->n_eq; c.src_head = &p.ctl->head_eq;
    c.buffer_is_debug = 0;                        // queued secondaries are not incident energy (mc_transport_debug's buffer is)
    launch_electron(p, c);
  }

  // Prologue on the caller's stream: zero the control blocks (and the internal grid), pack the phantom, fork the pipelines.
  int begin(void *workspace, size_t workspace_bytes, bool host_staging, const phantom_t &ph, long long *dose_acc, const mc_opts_t &o,
            uint64_t batch_, const char *who) {
    nvox = (size_t)ph.nx * ph.ny * ph.nz; batch = batch_;
    L = make_layout(batch, nvox, brick_count(ph.nx, ph.ny, ph.nz));
    if (!workspace || workspace_bytes < (host_staging ? L.host_total : L.total)) {
      char b[160]; snprintf(b, sizeof b, "%s: workspace missing or too small (see mc_workspace_bytes)", who);
      return fail(MC_E_WORKSPACE, b);
    }
    ws = (char *)workspace; us = (cudaStream_t)o.cuda_stream; flags = o.flags;
    eq_cap = o.debug_eq_cap ? std::min(o.debug_eq_cap, L.eq_cap) : L.eq_cap;
    dbg = (o.flags & MC_FLAG_STATS) || o.fingerprints;                        // stats and fingerprints live in the DBG variants,
    mode = dbg ? MODE_DBG : (o.com_index ? MODE_COM : MODE_PLAIN);            // the commissioning tally has its own
    timing = (o.flags & MC_FLAG_TIMING) != 0;
    npipe = o.pipelines > 0 ? o.pipelines : kMaxPipes;
    npipe = std::max(1, std::min(npipe, kMaxPipes));
    for (int p = 0; p < std::min(npipe, 2); ++p) if (npipe > 1 && !o.aux_streams[p]) npipe = 1;     // no streams given: serial
    if (npipe > 1 && (o.aux_streams[0] == o.aux_streams[1] || o.aux_streams[0] == o.cuda_stream || o.aux_streams[1] == o.cuda_stream))
      return fail(MC_E_INVALID_ARG, "aux_streams must be distinct from each other and from cuda_stream");
    long long *acc = dose_acc ? dose_acc : (long long *)(ws + L.acc);
    g = make_grid(ph, acc); g.vox = (const uint32_t *)(ws + L.vox);
    g.nbx = (ph.nx + 3) / 4; g.nby = (ph.ny + 3) / 4; g.nbricks = (unsigned)((size_t)g.nbx * g.nby * ((ph.nz + 3) / 4));
    g.nsx = (g.nbx + 3) / 4; g.nsy = (g.nby + 3) / 4; g.sbrick = (const uint32_t *)(ws + L.sbrick);
    g.brick = (const uint32_t *)(ws + L.brick); g.n_uniform = &((Control *)(ws + L.ctl[0]))->n_uniform_bricks;
    g.n_uniform_sb = &((Control *)(ws + L.ctl[0]))->n_uniform_sbricks; g.nsbricks = (unsigned)(g.nsx * g.nsy * (((ph.nz + 3) / 4 + 3) / 4));
    g.com_index = (const int *)o.com_index; g.com_dose = (unsigned long long *)o.com_dose; g.com_rows = o.com_rows;
    g.com_mask = (const uint32_t *)(ws + L.com_mask); g.com_coarse = (const uint32_t *)(ws + L.com_coarse);
    for (int p = 0; p < npipe; ++p) {
      Pipe &q = pipes[p];
      q.st = (npipe > 1 && p < 2) ? (cudaStream_t)o.aux_streams[p] : us; q.ctl = (Control *)(ws + L.ctl[p]);
      q.p0 = (float4 *)(ws + L.p0[p]); q.p1 = (float4 *)(ws + L.p1[p]); q.p2 = (uint32_t *)(ws + L.p2[p]);
      q.q0 = (float4 *)(ws + L.q0[p]); q.q1 = (float4 *)(ws + L.q1[p]); q.q2 = (uint32_t *)(ws + L.q2[p]);
      q.tile_count = (unsigned *)(ws + L.tile[p]); q.tile_cursor = q.tile_count + kTileBinsMax;
      q.eq.a = (float4 *)(ws + L.eq[p][0]); q.eq.b = (float4 *)(ws + L.eq[p][1]); q.eq.c = (uint4 *)(ws + L.eq[p][2]);
      q.eq.count = &q.ctl->n_eq; q.eq.cap = eq_cap;
      q.tm.on = timing; q.tm.st = q.st;
    }
    // Persistent grids fill every CTA slot except in one case: a phantom whose packed words + int64 grid (12 B per voxel)
    // do not fit L2, several pipelines and batches below 2^24.  There the launch tails are frequent and a grid of 0.75 leaves
    // slots in which the next pipeline's CTAs start while this kernel drains (C4, three pipelines: 72.8 against 73.8 ms per 2e8
    // at batch 2^22, 127 against 143 ms at 2^17).  Alone on the GPU a full grid is 8-11 % faster (C4 serial: 142.8 against
    // 159.0 ms per 4e8), and with batches of 2^24 still 1 % (140.5 against 141.9 ms): profiles/r2_ablation_c4.md.
    const bool big = 12.0 * (double)nvox > 110e6;
    init_blocks(big && npipe > 1 && batch < (1ull << 24) ? 0.75 : 1.0);
    { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev); }
    // Entry-tile ordering of every batch (the spatial inner loop): MC_FLAG_TILE_SORT.  Off by default:
    // measured on C4 it takes 10 % off the transport kernels' time and costs as much in the sort - photons
    // scatter 10-20 cm away from their entry tile.  Cubic tiles of 2^shift voxels, at most kTileBinsMax bins.
    tm = TileMap{};
    blocks_sample = 0;
    if ((o.flags & MC_FLAG_TILE_SORT) && !(o.flags & MC_FLAG_NO_TILE_SORT)) {
      int sh = 3;
      auto nt = [&](int n) { return ((n - 1) >> sh) + 1; };
      while ((long long)nt(ph.nx) * nt(ph.ny) * nt(ph.nz) > kTileBinsMax) ++sh;
      tm.shift = sh; tm.ntx = nt(ph.nx); tm.nty = nt(ph.ny); tm.nbins = tm.ntx * tm.nty * nt(ph.nz);
    }
    blocks_sample = persistent_blocks(k_sample, sizeof(unsigned) * tm.nbins, 1.0);      // (70 registers: 3 CTAs per SM)
    rhomax = pipes[0].ctl->rhomax;
    CUDA_TRY(cudaEventCreate(&ev0)); CUDA_TRY(cudaEventCreate(&ev1));
    CUDA_TRY(cudaEventRecord(ev0, us));
    CUDA_TRY(cudaMemsetAsync(ws, 0, L.zero_bytes, us));          // every pipeline's control block and entry-tile counters
    if (!dose_acc) CUDA_TRY(cudaMemsetAsync(acc, 0, 8 * nvox, us));
    tm_us.on = timing; tm_us.st = us;
    tm_us.begin(MC_K_AUX);
    k_pack_phantom<<<592, 256, 0, us>>>(ph.density, ph.material, nvox, (uint32_t *)(ws + L.vox), pipes[0].ctl);
    k_bricks<<<(g.nbricks + 63) / 64, 64, 0, us>>>(g.vox, g.nx, g.ny, g.nz, g.nbx, g.nby, g.nbricks, (uint32_t *)(ws + L.brick), pipes[0].ctl);
    { const int nbz = (ph.nz + 3) / 4; const unsigned nsb = (unsigned)(g.nsx * g.nsy * ((nbz + 3) / 4));
      k_sbricks<<<(nsb + 31) / 32, 32, 0, us>>>(g.brick, g.nbx, g.nby, nbz, g.nsx, g.nsy, nsb, (uint32_t *)(ws + L.sbrick), pipes[0].ctl); ++launches_us[MC_K_AUX]; }
    if (g.com_index) { k_com_mask<<<(unsigned)(((nvox + 31) / 32 + 255) / 256), 256, 0, us>>>(g.com_index, nvox, (uint32_t *)(ws + L.com_mask), (uint32_t *)(ws + L.com_coarse)); ++launches_us[MC_K_AUX]; }
    tm_us.end(MC_K_AUX); launches_us[MC_K_AUX] += 2;
    if (npipe > 1) {
      CUDA_TRY(cudaEventCreateWithFlags(&ev_fork, cudaEventDisableTiming));
      CUDA_TRY(cudaEventRecord(ev_fork, us));
      for (int p = 0; p < npipe; ++p) if (pipes[p].st != us) CUDA_TRY(cudaStreamWaitEvent(pipes[p].st, ev_fork, 0));
    }
    memset(&g_stats, 0, sizeof g_stats);
    return MC_OK;
  }

  // Enqueues every launch of histories [hb, he) of an N-history allocation of one beam.
  int run_beam(const psl_t *P, const beam_geom_t &beam, uint64_t N, uint64_t seed, uint64_t hb, uint64_t he, bool mixed) {
    xs.data = (const float *)P->d_xs; xs.x0 = (float)P->xs_x0; xs.inv_h = (float)(1.0 / P->xs_h); xs.n = kXsIntervals;
    std::vector<uint64_t> off(P->groups.size() + 1);
    allocate_host(*P, N, off.data());
    const uint64_t perm_a = mixed ? mixed_multiplier(N) : 0;
    SampleArgs sa{};
    sa.m = source_model(*P); sa.beam = beam_xf(beam); sa.seed = seed; round_keys(seed, sa.ks); sa.n_total = N; sa.perm_a = perm_a;
    for (size_t i = 0; i < off.size(); ++i) sa.off_g[i] = off[i];
    sa.fp = fp; sa.fp_base = fp_base; sa.compact = 1; sa.g = g; sa.stats = dbg ? 1 : 0;
    auto sample_batch = [&](Pipe &p, uint64_t first, uint64_t count) {
      if (p.started) { p.tm.begin(MC_K_AUX); k_next_batch<<<1, 1, 0, p.st>>>(p.ctl); p.tm.end(MC_K_AUX); ++p.launches[MC_K_AUX]; }
      p.started = true;                                   // (a pipeline's first batch finds the control block freshly zeroed)
      sa.first = first; sa.count = (unsigned)count; sa.p0 = p.p0; sa.p1 = p.p1; sa.ctl = p.ctl;
      sa.p2 = g.com_index ? p.p2 : nullptr;
      sa.tm = tm; sa.tile_count = tm.nbins ? p.tile_count : nullptr;
      p.tm.begin(MC_K_SAMPLE);
      const unsigned nblk = (unsigned)std::min<uint64_t>((count + 2 * kThreads - 1) / (2 * kThreads), (uint64_t)blocks_sample);     // persistent; a CTA takes 512 histories per iteration
      k_sample<<<nblk, kThreads, sizeof(unsigned) * tm.nbins, p.st>>>(sa);
      if (tm.nbins) {                                     // counting sort of the survivors by entry tile: counts -> cursors -> moves
        k_tile_scan<<<1, 1024, 0, p.st>>>(p.tile_count, p.tile_cursor, tm.nbins);
        ScatterArgs sc{};
        sc.g = g; sc.tm = tm; sc.p0 = p.p0; sc.p1 = p.p1; sc.p2 = sa.p2; sc.q0 = p.q0; sc.q1 = p.q1; sc.q2 = p.q2;
        sc.n_pb = &p.ctl->n_pb; sc.cursor = p.tile_cursor;
        const unsigned nsc = (unsigned)std::min<uint64_t>((count + kTileChunk - 1) / kTileChunk, (uint64_t)sms * 4);
        k_tile_scatter<<<nsc, kThreads, 2 * sizeof(unsigned) * tm.nbins, p.st>>>(sc);
        p.launches[MC_K_SAMPLE] += 2;
      }
      p.tm.end(MC_K_SAMPLE); ++p.launches[MC_K_SAMPLE];
    };
    auto photon_batch = [&](Pipe &p, uint64_t first) {   // the photons of the particle buffer, then every electron they queued
      TransportArgs a = base_args(p, seed, N, perm_a);
      a.src_kind = SRC_BUFFER; a.buffer_is_debug = 0; a.first = first; a.want_type = 0;
      a.src_count = &p.ctl->n_pb; a.src_head = &p.ctl->head_pb;
      launch_photon(p, a);
      drain_electrons(p, a);
    };
    auto electron_batch = [&](Pipe &p, uint64_t first, unsigned *head) {     // contamination electrons straight from the buffer
      TransportArgs a = base_args(p, seed, N, perm_a);
      a.src_kind = SRC_BUFFER; a.buffer_is_debug = 0; a.first = first; a.want_type = 1;
      a.src_count = &p.ctl->n_pb; a.src_head = head;
      launch_electron(p, a);
    };
    const int ne = P->n_ebin;
    if (!mixed) {
      // one sub-source type at a time, energy bins ascending, M histories per launch
      for (int s = 0; s < 3; ++s) {
        const uint64_t lo = std::max(hb, off[(size_t)s * ne]), hi = std::min(he, off[(size_t)(s + 1) * ne]);
        if (lo >= hi) continue;
        g_stats.n_hist[s] += hi - lo;
        // equal batches: ceil(n / batch) launches of the same size (a short last batch is mostly tail)
        const uint64_t nb = (hi - lo + batch - 1) / batch, even = std::min(batch, (((hi - lo + nb - 1) / nb) + kThreads - 1) / kThreads * kThreads);
        for (uint64_t first = lo; first < hi; first += even, ++task) {
          Pipe &p = pipes[task % npipe];
          sample_batch(p, first, std::min(even, hi - first));
          if (P->psr.particle_type[s] == 0) photon_batch(p, first);
          else electron_batch(p, first, &p.ctl->head_pb);
        }
      }
    } else {
      for (uint64_t first = hb; first < he; first += batch, ++task) {
        Pipe &p = pipes[task % npipe];
        sample_batch(p, first, std::min(batch, he - first));
        electron_batch(p, first, &p.ctl->head_pb_e);
        photon_batch(p, first);
      }
      if (hb == 0 && he == N) for (int s = 0; s < 3; ++s) g_stats.n_hist[s] += off[(size_t)(s + 1) * ne] - off[(size_t)s * ne];   // (not tracked per range)
    }
    CUDA_TRY(cudaGetLastError());
    return MC_OK;
  }

  // Joins the pipelines, converts (or only scans) the grid, synchronises once, folds the control blocks into g_stats.
  int end(const phantom_t &ph, double *dose_out, uint64_t n_norm, uint64_t n_run, const char *who) {
    for (int p = 0; p < npipe && npipe > 1; ++p) {
      if (pipes[p].st == us) continue;                      // (the third pipeline runs on the caller's stream itself)
      CUDA_TRY(cudaEventCreateWithFlags(&ev_join[p], cudaEventDisableTiming));
      CUDA_TRY(cudaEventRecord(ev_join[p], pipes[p].st));
      CUDA_TRY(cudaStreamWaitEvent(us, ev_join[p], 0));
    }
    tm_us.begin(MC_K_FINALISE);
    const double inv_vn = 1.0 / (ph.dx * ph.dy * ph.dz * (double)std::max<uint64_t>(1, n_norm));
    k_finalise<<<592, 256, 0, us>>>((const long long *)g.acc, ph.density, nvox, inv_vn, dose_out, pipes[0].ctl);
    tm_us.end(MC_K_FINALISE); ++launches_us[MC_K_FINALISE];
    CUDA_TRY(cudaEventRecord(ev1, us));
    CUDA_TRY(cudaGetLastError());
    Control hc[kMaxPipes];
    for (int p = 0; p < npipe; ++p) CUDA_TRY(cudaMemcpyAsync(&hc[p], pipes[p].ctl, sizeof(Control), cudaMemcpyDeviceToHost, us));
    CUDA_TRY(cudaStreamSynchronize(us));
    CUDA_TRY(cudaEventElapsedTime(&g_stats.ms_total, ev0, ev1));
    // fold the pipelines: kernel-class times add up (they overlap in wall time), counters and ledgers sum exactly
    tm_us.collect(g_stats.ms);
    Control &c = hc[0];
    for (int p = 0; p < npipe; ++p) {
      hc[p].n_accepted += hc[p].n_pb; hc[p].hw_eq = std::max(hc[p].hw_eq, hc[p].n_eq);      // what k_next_batch would have folded for the last batch
      float ms[5]; pipes[p].tm.collect(ms);
      for (int k = 0; k < 5; ++k) { g_stats.ms[k] += ms[k]; launches_us[k] += pipes[p].launches[k]; }
      if (p == 0) continue;
      for (int sl = 0; sl < kLedgerSlots; ++sl)
        for (int k = 0; k < 4; ++k) {
          unsigned __int128 a = ((unsigned __int128)c.ledger[sl][k][1] << 64) | c.ledger[sl][k][0];
          a += ((unsigned __int128)hc[p].ledger[sl][k][1] << 64) | hc[p].ledger[sl][k][0];
          c.ledger[sl][k][0] = (unsigned long long)a; c.ledger[sl][k][1] = (unsigned long long)(a >> 64);
        }
      for (int k = 0; k < ST_COUNT; ++k) c.stat[k] += hc[p].stat[k];
      c.hw_eq = std::max(c.hw_eq, hc[p].hw_eq);
      c.n_accepted += hc[p].n_accepted; c.n_missed += hc[p].n_missed; c.overflow |= hc[p].overflow; c.bad_input |= hc[p].bad_input;
    }
    mc_stats_t *s = &g_stats;
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
    s->n_deposits = c.stat[ST_DEPOSITS]; s->n_kahn_trials = c.stat[ST_KAHN]; s->n_deflections = c.stat[ST_DEFLECT];
    s->queue_high_water = c.hw_eq;
    for (int k = 0; k < 5; ++k) s->launches[k] = launches_us[k];
    s->n_jaw_rejected = n_run >= c.n_accepted + c.n_missed ? n_run - c.n_accepted - c.n_missed : 0;
    char b[200];
    if (c.overflow & 1u) { snprintf(b, sizeof b, "%s: the electron queue overflowed (capacity %u entries); use a larger batch workspace", who, eq_cap); return fail(MC_E_OVERFLOW, b); }
    if (c.overflow & 2u) { snprintf(b, sizeof b, "%s: a voxel's int64 accumulator wrapped (more than 2^63 quanta = 2.1e9 MeV in one voxel)", who); return fail(MC_E_OVERFLOW, b); }
    if (c.bad_input) { snprintf(b, sizeof b, "%s: a particle energy outside [0, 4096) MeV", who); return fail(MC_E_INVALID_ARG, b); }
    return MC_OK;
  }

  static uint64_t gcd_u64(uint64_t a, uint64_t b) { while (b) { uint64_t t = a % b; a = b; b = t; } return a; }
  // Mixed order (ablation): thread t handles history (a*t) mod N, a = smallest integer >= floor(0.618...N) coprime to N.
  static uint64_t mixed_multiplier(uint64_t N) {
    if (N < 3) return 1;
    uint64_t a = (uint64_t)(0.6180339887 * (double)N);
    if (a < 1) a = 1;
    while (gcd_u64(a, N) != 1) ++a;
    return a;
  }
};

constexpr uint64_t kMaxHistories = 1ull << 53;        // Eq. 3 is evaluated in double: N must be exactly representable

static int check_common(const psl_t *P, const phantom_t *ph, uint64_t N, uint64_t batch, const mc_opts_t *o, const char *who) {
  char b[200];
  if (!P || !phantom_ok(ph) || N == 0 || N > kMaxHistories || batch == 0 || batch > (1ull << 30)) {
    snprintf(b, sizeof b, "%s: invalid argument (null handle, bad phantom, n_histories outside [1, 2^53] or batch outside [1, 2^30])", who);
    return fail(MC_E_INVALID_ARG, b);
  }
  if (o->reserved || o->reserved2) { snprintf(b, sizeof b, "%s: reserved fields of mc_opts_t must be 0", who); return fail(MC_E_INVALID_ARG, b); }
  int dev = 0; CUDA_TRY(cudaGetDevice(&dev));
  if (dev != P->device) { snprintf(b, sizeof b, "%s: psl_t was built on device %d, the current device is %d", who, P->device, dev); return fail(MC_E_INVALID_ARG, b); }
  return MC_OK;
}

// The driver proper.  All pointers inside `ph` are DEVICE pointers here.
static int run_dose(const psl_t *P, const phantom_t *ph, const beam_geom_t *beam, uint64_t N, uint64_t seed, uint64_t batch,
                    double *dose_out, const mc_opts_t *opts, bool host_staging) {
  static const mc_opts_t kDefaults = {};
  if (!opts) opts = &kDefaults;
  if (!beam || (!dose_out && !opts->dose_acc)) return fail(MC_E_INVALID_ARG, "mc_dose: invalid argument (beam, or neither dose_out nor dose_acc)");
  if (int rc = check_common(P, ph, N, batch, opts, "mc_dose")) return rc;
  const bool ranged = (opts->flags & MC_FLAG_RANGE) != 0;
  const uint64_t hb = opts->history_begin, he = (ranged || opts->history_end) ? opts->history_end : N;
  if (hb > he || he > N) return fail(MC_E_INVALID_ARG, "mc_dose: history range outside [0, n_histories]");
  const bool mixed = opts->order == MC_ORDER_MIXED;
  if (mixed && (N >> 32)) return fail(MC_E_INVALID_ARG, "mc_dose: mixed order needs n_histories < 2^32");
  if (mixed && opts->fingerprints && (hb != 0 || he != N)) return fail(MC_E_INVALID_ARG, "mc_dose: mixed order + fingerprints needs the full range");
  if (opts->com_index) {
    if (!opts->com_dose || opts->com_rows < 1 || opts->com_cols != 2 * P->n_ebin * P->n_ring + P->n_ebin)
      return fail(MC_E_INVALID_ARG, "mc_dose: commissioning tally needs com_dose, com_rows >= 1 and com_cols = 2*n_ebin*n_ring + n_ebin");
    if (P->psr.particle_type[0] != 0 || P->psr.particle_type[1] != 0 || P->psr.particle_type[2] != 1)
      return fail(MC_E_INVALID_ARG, "mc_dose: the commissioning columns are defined for particle_type = {0, 0, 1} (two photon sub-sources, one electron sub-source)");
    if (mixed) return fail(MC_E_INVALID_ARG, "mc_dose: the commissioning tally runs in sorted order");
  }
  Session S;
  S.fp = (unsigned long long *)opts->fingerprints; S.fp_base = hb;
  if (int rc = S.begin(opts->workspace, opts->workspace_bytes, host_staging, *ph, (long long *)opts->dose_acc, *opts, batch, "mc_dose")) return rc;
  if (int rc = S.run_beam(P, *beam, N, seed, hb, he, mixed)) return rc;
  return S.end(*ph, dose_out, N, he - hb, "mc_dose");
}

}  // namespace pslmc

using namespace pslmc;

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

extern "C" size_t mc_workspace_bytes(const psl_t *, const phantom_t *ph, uint64_t batch) {
  if (!ph || ph->nx <= 0 || ph->ny <= 0 || ph->nz <= 0 || batch == 0 || batch > (1ull << 30)) return 0;
  return make_layout(batch, (size_t)ph->nx * ph->ny * ph->nz, brick_count(ph->nx, ph->ny, ph->nz)).total;
}
extern "C" size_t mc_host_workspace_bytes(const psl_t *, const phantom_t *ph, uint64_t batch) {
  if (!ph || ph->nx <= 0 || ph->ny <= 0 || ph->nz <= 0 || batch == 0 || batch > (1ull << 30)) return 0;
  return make_layout(batch, (size_t)ph->nx * ph->ny * ph->nz, brick_count(ph->nx, ph->ny, ph->nz)).host_total;
}

extern "C" int mc_dose(const psl_t *P, const phantom_t *ph, const beam_geom_t *beam, uint64_t n_histories, uint64_t seed,
                       uint64_t batch, double *dose_out, const mc_opts_t *opts) {
  return run_dose(P, ph, beam, n_histories, seed, batch, dose_out, opts, false);
}

extern "C" int mc_dose_host(const psl_t *P, const phantom_t *ph, const beam_geom_t *beam, uint64_t n_histories, uint64_t seed,
                            uint64_t batch, double *dose_out_host, const mc_opts_t *opts) {
  if (!ph || ph->nx <= 0 || ph->ny <= 0 || ph->nz <= 0 || !ph->density || !ph->material || !dose_out_host || !opts || batch == 0 || batch > (1ull << 30))
    return fail(MC_E_INVALID_ARG, "mc_dose_host: invalid argument (opts with a workspace is required)");
  const size_t nvox = (size_t)ph->nx * ph->ny * ph->nz;
  const Layout L = make_layout(batch, nvox, brick_count(ph->nx, ph->ny, ph->nz));
  if (!opts->workspace || opts->workspace_bytes < L.host_total) return fail(MC_E_WORKSPACE, "mc_dose_host: workspace missing or too small (see mc_host_workspace_bytes)");
  cudaStream_t st = (cudaStream_t)opts->cuda_stream;
  char *b = (char *)opts->workspace;
  CUDA_TRY(cudaMemcpyAsync(b + L.host_rho, ph->density, 4 * nvox, cudaMemcpyHostToDevice, st));
  CUDA_TRY(cudaMemcpyAsync(b + L.host_mat, ph->material, nvox, cudaMemcpyHostToDevice, st));
  phantom_t d = *ph; d.density = (const float *)(b + L.host_rho); d.material = (const uint8_t *)(b + L.host_mat);
  int rc = run_dose(P, &d, beam, n_histories, seed, batch, (double *)(b + L.host_dose), opts, true);
  if (rc) return rc;
  CUDA_TRY(cudaMemcpyAsync(dose_out_host, b + L.host_dose, 8 * nvox, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  return MC_OK;
}

extern "C" int mc_plan_dose(const psl_t *const *psls, const beam_geom_t *beams, int32_t n_beams, const phantom_t *ph,
                            uint64_t n_histories, uint64_t seed, uint64_t batch, double *dose_out, const mc_opts_t *opts,
                            uint64_t *n_beam_out) {
  static const mc_opts_t kDefaults = {};
  if (!opts) opts = &kDefaults;
  if (!psls || !beams || n_beams < 1 || (!dose_out && !opts->dose_acc)) return fail(MC_E_INVALID_ARG, "mc_plan_dose: invalid argument");
  if (opts->history_begin || opts->history_end || opts->fingerprints || opts->com_index || opts->order != MC_ORDER_SORTED || (opts->flags & MC_FLAG_RANGE))
    return fail(MC_E_INVALID_ARG, "mc_plan_dose: history ranges, fingerprints, mixed order and the commissioning tally are per-beam options (use mc_dose)");
  const int world = opts->shard_count > 0 ? opts->shard_count : 1, rank = opts->shard_count > 0 ? opts->shard_index : 0;
  if (rank < 0 || rank >= world) return fail(MC_E_INVALID_ARG, "mc_plan_dose: shard_index outside [0, shard_count)");
  for (int i = 0; i < n_beams; ++i) if (int rc = check_common(psls[i], ph, n_histories, batch, opts, "mc_plan_dose")) return rc;
  std::vector<uint64_t> n(n_beams);
  if (int rc = mc_plan_allocate(psls, n_beams, n_histories, n.data())) return rc;
  if (n_beam_out) std::copy(n.begin(), n.end(), n_beam_out);
  Session S;
  if (int rc = S.begin(opts->workspace, opts->workspace_bytes, false, *ph, (long long *)opts->dose_acc, *opts, batch, "mc_plan_dose")) return rc;
  uint64_t n_run = 0;
  for (int i = 0; i < n_beams; ++i) {
    // shard `rank` of beam i: the same contiguous split as binding.shard_range (n*r/world in 128-bit: n <= 2^53, world < 2^31)
    const uint64_t hb = (uint64_t)((unsigned __int128)n[i] * rank / world), he = (uint64_t)((unsigned __int128)n[i] * (rank + 1) / world);
    if (hb >= he) continue;
    if (int rc = S.run_beam(psls[i], beams[i], n[i], seed + (uint64_t)i, hb, he, false)) return rc;
    n_run += he - hb;
  }
  return S.end(*ph, dose_out, n_histories, n_run, "mc_plan_dose");
}

extern "C" int mc_stats(mc_stats_t *out) {
  if (!out) return fail(MC_E_INVALID_ARG, "mc_stats: null argument");
  *out = g_stats;
  return MC_OK;
}

// ---------------------------------------------------------------- parity / debug exports
extern "C" int mc_sample_debug(const psl_t *P, const beam_geom_t *beam, uint64_t first_history, uint64_t count,
                               uint64_t n_histories, uint64_t seed, float *soa_out, void *cuda_stream) {
  if (!P || !beam || n_histories == 0 || n_histories > kMaxHistories || first_history + count > n_histories || count > 0x7fffffffull)
    return fail(MC_E_INVALID_ARG, "mc_sample_debug: invalid argument");
  if (count == 0) return MC_OK;
  if (!soa_out) return fail(MC_E_INVALID_ARG, "mc_sample_debug: soa_out is null");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  std::vector<uint64_t> off(P->groups.size() + 1);
  allocate_host(*P, n_histories, off.data());
  SampleArgs sa{};
  sa.m = source_model(*P); sa.beam = beam_xf(*beam);
  for (size_t i = 0; i < off.size(); ++i) sa.off_g[i] = off[i];
  sa.seed = seed; round_keys(seed, sa.ks); sa.first = first_history; sa.n_total = n_histories; sa.perm_a = 0; sa.count = (unsigned)count;
  sa.p0 = (float4 *)soa_out; sa.p1 = (float4 *)soa_out + count; sa.ctl = nullptr; sa.fp = nullptr; sa.compact = 0;
  int sms = 1; cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, P->device);
  k_sample<<<(unsigned)std::min<uint64_t>((count + 2 * kThreads - 1) / (2 * kThreads), (uint64_t)sms * 8), kThreads, 0, st>>>(sa);
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaStreamSynchronize(st));
  return MC_OK;
}

extern "C" int mc_transport_debug(const phantom_t *ph, int32_t particle_type, const float *soa_in, uint64_t first_history,
                                  uint64_t count, uint64_t seed, const mc_opts_t *opts) {
  if (!phantom_ok(ph) || !soa_in || !opts || !opts->dose_acc || (particle_type != 0 && particle_type != 1) || count > (1ull << 30))
    return fail(MC_E_INVALID_ARG, "mc_transport_debug: invalid argument (opts->dose_acc is required)");
  memset(&g_stats, 0, sizeof g_stats);
  if (count == 0) return MC_OK;
  Session S;
  mc_opts_t o = *opts; o.flags |= MC_FLAG_STATS; o.pipelines = 1;
  S.fp = (unsigned long long *)opts->fingerprints; S.fp_base = first_history;
  if (int rc = S.begin(opts->workspace, opts->workspace_bytes, false, *ph, (long long *)opts->dose_acc, o, count, "mc_transport_debug")) return rc;
  Pipe &p = S.pipes[0];
  // cross-section nodes for energies up to 64 MeV (debug entry: any energy below that), in the workspace
  const double x0 = std::log2(0.045), hh = (std::log2(64.0 * 1.001) - x0) / kXsIntervals;
  float *nodes = (float *)(S.ws + S.L.xs);
  k_build_xs<<<(kXsIntervals + 256) / 256, 256, 0, p.st>>>(nullptr, nodes, x0, hh, kXsIntervals);
  S.xs.data = nodes; S.xs.x0 = (float)x0; S.xs.inv_h = (float)(1.0 / hh); S.xs.n = kXsIntervals;
  // the caller's planes stand in for the particle buffer; n_pb = count
  const unsigned cnt = (unsigned)count;
  CUDA_TRY(cudaMemcpyAsync(&p.ctl->n_pb, &cnt, sizeof cnt, cudaMemcpyHostToDevice, p.st));
  TransportArgs a = S.base_args(p, seed, first_history + count, 0);
  a.p0 = (const float4 *)soa_in; a.p1 = (const float4 *)soa_in + count; a.p2 = nullptr;
  a.src_kind = SRC_BUFFER; a.buffer_is_debug = 1; a.first = first_history; a.want_type = particle_type;
  a.src_count = &p.ctl->n_pb; a.src_head = &p.ctl->head_pb;
  if (particle_type == 0) { S.launch_photon(p, a); S.drain_electrons(p, a); }
  else S.launch_electron(p, a);
  k_next_batch<<<1, 1, 0, p.st>>>(p.ctl);
  return S.end(*ph, nullptr, 1, 0, "mc_transport_debug");
}

// (debug probe: allocates its own few KB of device memory - not on the hot path)
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
  const double x0 = std::log2(0.045), hh = (std::log2(e_max * 1.001) - x0) / kXsIntervals;
  k_build_xs<<<(kXsIntervals + 256) / 256, 256>>>((const Control *)(d + o_ctl), (float *)(d + o_xs), x0, hh, kXsIntervals);
  XsTable xs{(const float *)(d + o_xs), (float)x0, (float)(1.0 / hh), kXsIntervals};
  k_xs_debug<<<(unsigned)((n + 255) / 256), 256>>>(xs, (const float *)(d + o_e), n, (float *)(d + o_out));
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaMemcpy(out_host, d + o_out, 12 * n, cudaMemcpyDeviceToHost));
  cudaFree(d);
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
