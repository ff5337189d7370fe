// stag_ctx.cu — context, options, sizes, error strings of libstag_b200.so.
#include <cstdlib>
#include <cstring>
#include <cxxabi.h>
#include <new>
#include <string>

#include "stag_cg.cuh"

using namespace stag;

extern "C" int stag_ctx_create(const int L[4], stag_ctx **out) {
    if (!L || !out) return STAG_ERR_BADARG;
    long long V = 1;
    for (int mu = 0; mu < 4; ++mu) {
        if (L[mu] < 2 || (L[mu] & 1)) return STAG_ERR_BADARG;
        V *= L[mu];
        if (V >= (1ll << 31)) return STAG_ERR_UNSUPPORTED;
    }
    stag_ctx *c = new (std::nothrow) stag_ctx();
    if (!c) return STAG_ERR_CUDA;
    std::memset(&c->g, 0, sizeof(c->g));
    std::memset(&c->opt, 0, sizeof(c->opt));
    std::memset(c->slots, 0, sizeof(c->slots));
    c->nklog = 0; c->prof_iters = 0;
    Geom &g = c->g;
    for (int mu = 0; mu < 4; ++mu) g.L[mu] = L[mu];
    g.Lh0 = L[0] / 2;
    g.V = (int)V;
    g.Vh = (int)(V / 2);
    g.dLh0.init((uint32_t)g.Lh0);
    g.dL1.init((uint32_t)L[1]);
    g.dL2.init((uint32_t)L[2]);
    c->opt.dslash_block = 128;
    c->opt.dslash_regs = 0;
    c->opt.dslash_ctas_per_sm = 0;   // 0 = one CTA per 'dslash_block' sites (non-persistent)
    c->opt.dslash_pipe = 1;
    c->opt.cg_check_every = 16;
    c->opt.cg_graph = 1;
    c->opt.cg_freeze = 1;
    c->opt.cg_ctas_per_sm = 8;
    c->opt.cg_persistent = 1;
    c->opt.cg_persistent_threads = 0;
    c->opt.cg_resident_slices = 3;
    c->opt.cg_mixed_reliable = 1;
    c->opt.cg_mixed_delta_inv = 10;
    c->opt.cg_mixed_fp64_from = 3;
    c->opt.cg_l2_keep_mb = 64;
    c->opt.cg_fill = 1;
    c->opt.cg_nbflags = 1;
    c->opt.cg_single_reduction = 1;
    bool ok = cudaGetDevice(&c->device) == cudaSuccess &&
              cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, c->device) == cudaSuccess;
    for (int i = 0; i < kSlots && ok; ++i) {
        Slot &s = c->slots[i];
        ok = cudaHostAlloc((void **)&s.pinned_flags, 512, cudaHostAllocMapped) == cudaSuccess &&
             cudaHostAlloc(&s.pinned_info, sizeof(CgState), cudaHostAllocDefault) == cudaSuccess &&
             cudaEventCreateWithFlags(&s.ev[0], cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&s.ev[1], cudaEventDisableTiming) == cudaSuccess;
    }
    if (!ok) {
        cudaGetLastError();
        stag_ctx_destroy(c);
        return STAG_ERR_CUDA;
    }
    *out = c;
    return STAG_OK;
}

extern "C" void stag_ctx_destroy(stag_ctx *ctx) {
    if (!ctx) return;
    for (int i = 0; i < kSlots; ++i) {
        Slot &s = ctx->slots[i];
        if (s.gexec) cudaGraphExecDestroy(s.gexec);
        if (s.ev[0]) cudaEventDestroy(s.ev[0]);
        if (s.ev[1]) cudaEventDestroy(s.ev[1]);
        if (s.pinned_flags) cudaFreeHost(s.pinned_flags);
        if (s.pinned_info) cudaFreeHost(s.pinned_info);
    }
    delete ctx;
}

extern "C" const char *stag_strerror(int err) {
    switch (err) {
        case STAG_OK: return "ok";
        case STAG_ERR_BADARG: return "bad argument";
        case STAG_ERR_UNSUPPORTED: return "unsupported request";
        case STAG_ERR_CUDA: return "CUDA runtime error";
        case STAG_ERR_NOT_SU3: return "links are not SU(3): 12-real reconstruction impossible";
        case STAG_ERR_NOTCONV: return "multi-shift CG did not converge";
        case STAG_ERR_BREAKDOWN: return "multi-shift CG breakdown (<p,Ap> <= 0 or NaN)";
        case STAG_ERR_SCRATCH_LIMIT:
            return "problem too large for the built-in scratch of stag_fermion_force_static (8 MiB): "
                   "use stag_fermion_force with a workspace";
        default: return "unknown error";
    }
}

static int *option_slot(Options &o, const char *key) {
    if (!key) return nullptr;
    if (!std::strcmp(key, "dslash_block")) return &o.dslash_block;
    if (!std::strcmp(key, "dslash_regs")) return &o.dslash_regs;
    if (!std::strcmp(key, "dslash_ctas_per_sm")) return &o.dslash_ctas_per_sm;
    if (!std::strcmp(key, "dslash_pipe")) return &o.dslash_pipe;
    if (!std::strcmp(key, "cg_check_every")) return &o.cg_check_every;
    if (!std::strcmp(key, "cg_graph")) return &o.cg_graph;
    if (!std::strcmp(key, "cg_freeze")) return &o.cg_freeze;
    if (!std::strcmp(key, "cg_ctas_per_sm")) return &o.cg_ctas_per_sm;
    if (!std::strcmp(key, "cg_persistent")) return &o.cg_persistent;
    if (!std::strcmp(key, "cg_persistent_threads")) return &o.cg_persistent_threads;
    if (!std::strcmp(key, "cg_resident_slices")) return &o.cg_resident_slices;
    if (!std::strcmp(key, "cg_mixed_reliable")) return &o.cg_mixed_reliable;
    if (!std::strcmp(key, "cg_mixed_delta_inv")) return &o.cg_mixed_delta_inv;
    if (!std::strcmp(key, "cg_mixed_fp64_from")) return &o.cg_mixed_fp64_from;
    if (!std::strcmp(key, "cg_l2_keep_mb")) return &o.cg_l2_keep_mb;
    if (!std::strcmp(key, "cg_fill")) return &o.cg_fill;
    if (!std::strcmp(key, "cg_nbflags")) return &o.cg_nbflags;
    if (!std::strcmp(key, "cg_single_reduction")) return &o.cg_single_reduction;
    if (!std::strcmp(key, "cg_profile")) return &o.cg_profile;
    return nullptr;
}

extern "C" int stag_set_option(stag_ctx *ctx, const char *key, int value) {
    if (!ctx) return STAG_ERR_BADARG;
    int *slot = option_slot(ctx->opt, key);
    if (!slot) return STAG_ERR_BADARG;
    if (slot == &ctx->opt.dslash_block && value != 64 && value != 128 && value != 256)
        return STAG_ERR_BADARG;
    if (slot == &ctx->opt.dslash_regs && value != 0 && value != 64 && value != 128 && value != 255)
        return STAG_ERR_BADARG;
    if (slot == &ctx->opt.cg_check_every && value < 1) return STAG_ERR_BADARG;
    if (slot == &ctx->opt.cg_persistent_threads && value != 0 && value != 256 && value != 512 && value != 1024) return STAG_ERR_BADARG;
    if (slot == &ctx->opt.cg_mixed_delta_inv && value < 2) return STAG_ERR_BADARG;
    if (slot == &ctx->opt.cg_mixed_fp64_from && (value < 0 || value > STAG_MAX_SHIFTS + 1)) return STAG_ERR_BADARG;
    if (slot == &ctx->opt.cg_mixed_reliable && (value < 0 || value > 2)) return STAG_ERR_BADARG;
    if (slot == &ctx->opt.cg_resident_slices && (value < 0 || value > 3)) return STAG_ERR_BADARG;
    if (slot == &ctx->opt.cg_ctas_per_sm && (value < 1 || value > 16)) return STAG_ERR_BADARG;
    if (slot == &ctx->opt.cg_l2_keep_mb && (value < 0 || value > 1024)) return STAG_ERR_BADARG;
    if ((slot == &ctx->opt.cg_fill || slot == &ctx->opt.cg_nbflags || slot == &ctx->opt.cg_single_reduction || slot == &ctx->opt.cg_profile) &&
        (value < 0 || value > 1)) return STAG_ERR_BADARG;
    if (slot == &ctx->opt.dslash_ctas_per_sm && (value < 0 || value > 32)) return STAG_ERR_BADARG;
    *slot = value;
    return STAG_OK;
}

extern "C" int stag_get_option(const stag_ctx *ctx, const char *key, int *value) {
    if (!ctx || !value) return STAG_ERR_BADARG;
    int *slot = option_slot(const_cast<stag_ctx *>(ctx)->opt, key);
    if (!slot) return STAG_ERR_BADARG;
    *value = *slot;
    return STAG_OK;
}

// ---- sizes ------------------------------------------------------------------------------------
extern "C" size_t stag_gauge_canonical_bytes(const stag_ctx *ctx) {
    return ctx ? (size_t)ctx->g.V * 4 * 18 * sizeof(double) : 0;
}
extern "C" size_t stag_gauge_packed_bytes(const stag_ctx *ctx, int prec, int recon) {
    if (!ctx || !valid_prec(prec) || !valid_recon(recon)) return 0;
    return (size_t)16 * ctx->g.Vh * link_bytes_per_site(prec, recon);   // 2 parities x 8 directions
}
extern "C" size_t stag_vector_canonical_bytes(const stag_ctx *ctx) {
    return ctx ? (size_t)ctx->g.Vh * 6 * sizeof(double) : 0;
}
extern "C" size_t stag_vector_bytes(const stag_ctx *ctx, int prec) {
    if (!ctx || !valid_prec(prec)) return 0;
    return (size_t)ctx->g.Vh * vec_bytes_per_site(prec);
}
extern "C" size_t stag_cg_workspace_bytes(const stag_ctx *ctx, int prec, int nshift) {
    if (!ctx || !valid_prec(prec) || nshift < 1 || nshift > STAG_MAX_SHIFTS) return 0;
    return cg_workspace_layout(ctx, prec, nshift, nullptr);
}
extern "C" size_t stag_host_scratch_bytes(const stag_ctx *ctx, int prec, int nshift) {
    if (!ctx || !valid_prec(prec) || nshift < 0 || nshift > STAG_MAX_SHIFTS) return 0;
    const size_t canon = align256(stag_vector_canonical_bytes(ctx));
    const size_t vec = align256(stag_vector_bytes(ctx, prec));
    if (nshift == 0) return canon + 2 * vec;                       // canonical staging, in, out
    // canonical staging, b, y, x[nshift], CG workspace
    return canon + 2 * vec + align256((size_t)nshift * stag_vector_bytes(ctx, prec)) +
           align256(cg_workspace_layout(ctx, prec, nshift, nullptr));
}

// ---- measurement aids -------------------------------------------------------------------------------
extern "C" int stag_kernel_log_reset(const stag_ctx *ctx) {
    if (!ctx) return STAG_ERR_BADARG;
    std::lock_guard<std::mutex> lk(ctx->mu);          // log_kernel of a running call takes the same lock
    ctx->nklog = 0;
    return STAG_OK;
}

extern "C" int stag_kernel_log(const stag_ctx *ctx, char *buf, size_t nbytes) {
    if (!ctx || !buf || nbytes == 0) return STAG_ERR_BADARG;
    std::string out;
    const void *funcs[32];
    int n = 0;
    {
        std::lock_guard<std::mutex> lk(ctx->mu);
        n = ctx->nklog;
        for (int i = 0; i < n; ++i) funcs[i] = ctx->klog[i];
    }
    for (int i = 0; i < n; ++i) {
        const char *mangled = nullptr;
        if (cudaFuncGetName(&mangled, funcs[i]) != cudaSuccess || !mangled) { cudaGetLastError(); continue; }
        int status = 0;
        char *dem = abi::__cxa_demangle(mangled, nullptr, nullptr, &status);
        out += (status == 0 && dem) ? dem : mangled;
        out += '\n';
        std::free(dem);
    }
    if (out.size() + 1 > nbytes) return STAG_ERR_BADARG;
    std::memcpy(buf, out.c_str(), out.size() + 1);
    return n;
}

extern "C" int stag_cg_profile(const stag_ctx *ctx, double us_per_launch[4], int *iterations) {
    if (!ctx || !us_per_launch || !iterations) return STAG_ERR_BADARG;
    std::lock_guard<std::mutex> lk(ctx->mu);
    for (int j = 0; j < 4; ++j) us_per_launch[j] = ctx->prof_us[j];
    *iterations = ctx->prof_iters;
    return STAG_OK;
}
