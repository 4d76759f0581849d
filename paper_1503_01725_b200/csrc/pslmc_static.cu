// pslmc_static.cu — mc_dose_static: mc_dose for callers that may not allocate device memory (CUDA graph capture
// around the call site, serving loops, harnesses that forbid cudaMalloc).  The workspace mc_dose takes from its
// caller is here a file-scope __device__ array of MC_STATIC_WORKSPACE_BYTES: every GPU that loads the library
// holds it until the process exits.  Nothing else differs: the same Session, the same kernels, the same bits.
#include "pslmc_host.h"

#include <cstdio>
#include <mutex>

namespace pslmc {

// The scratch.  In host code `g_static_workspace` is only the host-side stand-in of the symbol, never a device
// address: the address comes from cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) unsigned char g_static_workspace[MC_STATIC_WORKSPACE_BYTES];

constexpr int kMaxDevices = 64;
static std::mutex g_static_mutex;
static void *g_static_ptr[kMaxDevices];          // per device ordinal, filled on first use

static int static_workspace(void **out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(MC_E_CUDA, std::string("mc_dose_static: cudaGetDevice failed: ") + cudaGetErrorString(e));
  if (dev < 0 || dev >= kMaxDevices) return fail(MC_E_INVALID_ARG, "mc_dose_static: device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (!g_static_ptr[dev]) {
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, g_static_workspace);
    if (e != cudaSuccess || !p)
      return fail(MC_E_CUDA, std::string("mc_dose_static: cudaGetSymbolAddress failed: ") + cudaGetErrorString(e));
    g_static_ptr[dev] = p;
  }
  *out = g_static_ptr[dev];
  return MC_OK;
}

}  // namespace pslmc

using namespace pslmc;

extern "C" size_t mc_static_workspace_bytes(void) { return (size_t)MC_STATIC_WORKSPACE_BYTES; }

extern "C" int mc_dose_static(const psl_t *psl, const phantom_t *ph, const beam_geom_t *beam, uint64_t n_histories,
                              uint64_t seed, uint64_t batch, double *dose_out, const mc_opts_t *opts) {
  if (!opts) return fail(MC_E_INVALID_ARG, "mc_dose_static: opts is NULL");
  if (opts->workspace || opts->workspace_bytes)
    return fail(MC_E_INVALID_ARG, "mc_dose_static: opts->workspace must be NULL (the scratch is the library's static array)");
  const size_t need = mc_workspace_bytes(psl, ph, batch);
  if (need == 0) return fail(MC_E_INVALID_ARG, "mc_dose_static: bad phantom or batch");
  if (need > (size_t)MC_STATIC_WORKSPACE_BYTES) {
    char b[256];
    snprintf(b, sizeof b, "mc_dose_static: this phantom and batch need %zu bytes of scratch, the static array holds %zu "
             "(MC_STATIC_WORKSPACE_BYTES): use a smaller batch, or mc_dose with a caller workspace",
             need, (size_t)MC_STATIC_WORKSPACE_BYTES);
    return fail(MC_E_WORKSPACE, b);
  }
  void *ws = nullptr;
  if (int rc = static_workspace(&ws)) return rc;
  mc_opts_t o = *opts;
  o.workspace = ws; o.workspace_bytes = (size_t)MC_STATIC_WORKSPACE_BYTES;
  return mc_dose(psl, ph, beam, n_histories, seed, batch, dose_out, &o);      // zeroes what must start at zero itself
}
