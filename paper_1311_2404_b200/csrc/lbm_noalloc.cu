// lbm_noalloc.cu -- lbm_step_noalloc: the whole path in ONE call that allocates nothing.
//
// Some callers cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses
// that forbid it) and cannot hand the library a workspace either.  For them the workspace of a
// context -- double-buffered distribution store, node-type / link encoding, Shan-Chen fields -- lives
// in the file-scope device array below, of a fixed, modest size.  Every GPU that loads the library
// holds the array until the process exits.  The entry point builds a context inside it, runs
// set_geometry -> set_distributions -> step(n) -> get_distributions through the ordinary C ABI (the
// same kernels as every other call), and destroys the context again; it calls no cudaMalloc, cudaFree,
// stream / graph creation or other allocating routine (graph replay is switched off for this context).
#include "lbm_impl.cuh"

#include <mutex>

namespace {

// 64 MiB: D3Q19 fp32 up to 64^3 nodes (174 B of workspace per node), D3Q19 fp64 up to 48^3.
constexpr size_t NOALLOC_MAX_BYTES = (size_t)LBM_NOALLOC_MAX_BYTES;
static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_MAX_BYTES];

// In host code `g_noalloc_scratch` is a host-side stand-in, not a device address: the address the
// kernels may use comes from cudaGetSymbolAddress, asked once per device with that device current.
constexpr int MAX_DEVICES = 64;
std::mutex g_lock;
void *g_scratch_ptr[MAX_DEVICES];

thread_local char g_noalloc_err[256] = "";

int noalloc_fail(int code, const char *fmt, const char *detail = "") {
    snprintf(g_noalloc_err, sizeof g_noalloc_err, fmt, detail);
    return code;
}

int scratch_for_current_device(void **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return noalloc_fail(LBM_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= MAX_DEVICES) return noalloc_fail(LBM_EUNSUPPORTED, "device ordinal beyond %s", "63");
    std::lock_guard<std::mutex> hold(g_lock);
    if (!g_scratch_ptr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return noalloc_fail(LBM_ECUDA, "cudaGetSymbolAddress(scratch): %s", cudaGetErrorString(e));
        }
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return LBM_OK;
}

}  // namespace

#define LBM_API extern "C" __attribute__((visibility("default")))

LBM_API int lbm_step_noalloc(const lbm_params *p, const uint8_t *d_mask, const void *d_f_in, void *d_f_out, int n,
                             void *cuda_stream) {
    g_noalloc_err[0] = 0;
    size_t need = 0;
    if (int rc = lbm_workspace_bytes(p, &need)) return noalloc_fail(rc, "%s", lbm_last_error(nullptr));
    if (!d_f_in || !d_f_out) return noalloc_fail(LBM_EINVAL, "d_f_in / d_f_out is %s", "NULL");
    if (n < 0) return noalloc_fail(LBM_EINVAL, "n %s", "< 0");
    if (need > NOALLOC_MAX_BYTES) {
        char msg[160];
        snprintf(msg, sizeof msg, "this lattice needs %zu bytes of scratch, the static maximum of lbm_step_noalloc is %zu (LBM_NOALLOC_MAX_BYTES)",
                 need, NOALLOC_MAX_BYTES);
        return noalloc_fail(LBM_EINVAL, "%s", msg);
    }
    if (p->store != LBM_STORE_AB) return noalloc_fail(LBM_EUNSUPPORTED, "lbm_step_noalloc runs the %s store only", "AB");
    void *scratch = nullptr;
    if (int rc = scratch_for_current_device(&scratch)) return rc;
    lbm_ctx *c = nullptr;
    // lbm_create clears the node-type and link arrays (the array keeps the last call's contents);
    // lbm_set_geometry clears its counter; every other region is written before it is read.
    if (int rc = lbm_create(p, scratch, NOALLOC_MAX_BYTES, cuda_stream, &c)) return noalloc_fail(rc, "%s", lbm_last_error(nullptr));
    c->no_graph = true;  // graph capture / instantiation would create a stream and allocate
    const size_t comp_bytes = (size_t)c->Q * (size_t)c->g.N * c->rs;
    int rc = LBM_OK;
    if (d_mask) rc = lbm_set_geometry(c, d_mask);
    for (int s = 0; s < c->ncomp && rc == LBM_OK; s++)
        rc = lbm_set_distributions(c, s, static_cast<const char *>(d_f_in) + s * comp_bytes);
    if (rc == LBM_OK) rc = lbm_step(c, n);
    for (int s = 0; s < c->ncomp && rc == LBM_OK; s++)
        rc = lbm_get_distributions(c, s, static_cast<char *>(d_f_out) + s * comp_bytes);
    if (rc != LBM_OK) noalloc_fail(rc, "%s", lbm_last_error(c));
    lbm_destroy(c);  // host object only: nothing was created on the device
    return rc;
}

LBM_API const char *lbm_noalloc_last_error(void) { return g_noalloc_err; }
