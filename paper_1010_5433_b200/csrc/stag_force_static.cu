// stag_force_static.cu — stag_fermion_force_static: the fermion force (N4, stag_force.cu; PAPER.md:25, :87,
// :93) for callers that cannot give it a workspace.
//
// Who needs this.  stag_fermion_force needs nshift odd-site vectors of scratch (w_i = D_oe x_i) and, like every
// call of this library, expects the caller to bring that memory.  Some callers have nothing to bring: a force
// routine called from inside somebody else's integrator is handed the x_i and the force array and nothing else;
// the host program may have given all device memory to its own pool at start-up, so a cudaMalloc from in here
// fails or takes memory the host counted on; and cudaMalloc / cudaFree synchronise the whole device, which a
// molecular-dynamics loop that keeps several streams busy cannot afford once per force evaluation.  For those
// callers the scratch lives in the library image itself: a fixed array in device global memory, present on every
// GPU that loads libstag_b200.so, from load until the process ends.
//
// What it costs.  STAG_FORCE_STATIC_BYTES (8 MiB) of every such GPU, used or not, and a hard size limit:
// stag_force_workspace_bytes(ctx, prec, nshift) must not exceed it (16^3 x 4 with 16 fp64 shifts is 6 MiB;
// 32^3 x 8 with 16 shifts is 96 MiB and is refused with STAG_ERR_SCRATCH_LIMIT).  There is ONE array per GPU:
// two calls that may run at the same time on the same GPU (different streams, different host threads, different
// contexts) write the same bytes and corrupt each other.  Order them on one stream or with events.
//
// The kernels are the ones stag_fermion_force launches; only the address of the scratch differs.
#include <mutex>

#include "stag_common.cuh"

namespace {

// The scratch.  Device code could name it directly; the host cannot: on the host `force_scratch` is only a
// handle for the runtime's symbol table, not an address a kernel may be given.  scratch_address() asks the
// runtime for the real device address, once per GPU.
static __device__ __align__(256) unsigned char force_scratch[STAG_FORCE_STATIC_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
void *g_scratch_addr[kMaxDevices];        // device address of force_scratch on GPU d, nullptr = not asked yet

// Device address of force_scratch on GPU `device`, which must be the current device.  The first call for a GPU
// is the set-up: it makes the runtime load this library's device code on that GPU (which is when the array comes
// to exist there) and look the symbol up; later calls read the cached pointer.
int scratch_address(int device, void **out) {
    if (device >= 0 && device < kMaxDevices) {
        std::lock_guard<std::mutex> lk(g_mu);
        if (!g_scratch_addr[device]) {
            void *p = nullptr;
            if (cudaGetSymbolAddress(&p, force_scratch) != cudaSuccess || !p) {
                cudaGetLastError();
                return STAG_ERR_CUDA;
            }
            g_scratch_addr[device] = p;
        }
        *out = g_scratch_addr[device];
        return STAG_OK;
    }
    void *p = nullptr;                    // more GPUs than the cache holds: look it up every time
    if (cudaGetSymbolAddress(&p, force_scratch) != cudaSuccess || !p) {
        cudaGetLastError();
        return STAG_ERR_CUDA;
    }
    *out = p;
    return STAG_OK;
}

}  // namespace

extern "C" size_t stag_fermion_force_static_max_bytes(void) { return (size_t)STAG_FORCE_STATIC_BYTES; }

extern "C" int stag_fermion_force_static(const stag_ctx *ctx, const void *packed, int prec, int recon, int nshift,
                                         const double *host_residues, const void *x_even, double *dev_force,
                                         int accumulate, void *stream) {
    if (!ctx || !packed || !host_residues || !x_even || !dev_force) return STAG_ERR_BADARG;
    // 0 = bad prec / nshift (the same rule stag_fermion_force applies)
    const size_t need = stag_force_workspace_bytes(ctx, prec, nshift);
    if (need == 0) return STAG_ERR_BADARG;
    if (need > (size_t)STAG_FORCE_STATIC_BYTES) return STAG_ERR_SCRATCH_LIMIT;
    // the array that must be used is the one on the GPU the context (and its buffers) belongs to, and the
    // runtime answers for the current GPU only
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess) { cudaGetLastError(); return STAG_ERR_CUDA; }
    if (cur != ctx->device) return STAG_ERR_BADARG;
    void *scratch = nullptr;
    const int rc = scratch_address(cur, &scratch);
    if (rc) return rc;
    // Nothing in the scratch has to start at zero: the D_oe launch writes every byte the force kernel reads
    // (all nshift vectors, every odd site) before that kernel starts on the same stream, so whatever an earlier
    // call — other lattice, precision or shift count — left behind is never read.
    return stag_fermion_force(ctx, packed, prec, recon, nshift, host_residues, x_even, dev_force, accumulate,
                              scratch, stream);
}
