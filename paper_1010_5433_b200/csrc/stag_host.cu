// stag_host.cu — the same calls on HOST buffers in canonical fp64 format: the end-to-end path a
// caller without device buffers uses (host<->device copies inside; PAPER.md:65 is why the paper
// avoids this inside a trajectory).  No arithmetic here: copy, convert, call, copy.
#include "stag_cg.cuh"

using namespace stag;

extern "C" int stag_dslash_host(const stag_ctx *ctx, const void *packed, int prec, int recon,
                                int out_parity, const double *host_in, double *host_out,
                                void *dev_scratch, void *stream) {
    if (!ctx || !packed || !host_in || !host_out || !dev_scratch) return STAG_ERR_BADARG;
    if (!valid_prec(prec) || !valid_recon(recon) || (out_parity != 0 && out_parity != 1))
        return STAG_ERR_BADARG;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t cbytes = stag_vector_canonical_bytes(ctx);
    const size_t canon_sz = align256(cbytes), vec_sz = align256(stag_vector_bytes(ctx, prec));
    char *s = static_cast<char *>(dev_scratch);
    double *canon = reinterpret_cast<double *>(s);
    void *vin = s + canon_sz, *vout = s + canon_sz + vec_sz;
    STAG_CUDA_OK(cudaMemcpyAsync(canon, host_in, cbytes, cudaMemcpyHostToDevice, st));
    int rc = stag_vector_pack(ctx, canon, vin, prec, st);
    if (rc) return rc;
    rc = dslash_dispatch(ctx, packed, prec, recon, vin, vout, out_parity, st);
    if (rc) return rc;
    rc = stag_vector_unpack(ctx, vout, prec, canon, st);
    if (rc) return rc;
    STAG_CUDA_OK(cudaMemcpyAsync(host_out, canon, cbytes, cudaMemcpyDeviceToHost, st));
    STAG_CUDA_OK(cudaStreamSynchronize(st));
    return STAG_OK;
}

extern "C" int stag_mshift_cg_host(const stag_ctx *ctx, const void *packed, int prec, int recon,
                                   const double *host_b, double mass, int nshift,
                                   const double *host_shifts, const double *host_residues,
                                   double residue0, double stop, int maxiter, double *host_x,
                                   double *host_y, void *dev_scratch, stag_cg_info *info,
                                   void *stream) {
    if (!ctx || !host_b || !host_x || !dev_scratch) return STAG_ERR_BADARG;
    if (!valid_prec(prec) || nshift < 1 || nshift > STAG_MAX_SHIFTS) return STAG_ERR_BADARG;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t cbytes = stag_vector_canonical_bytes(ctx);
    const size_t canon_sz = align256(cbytes), vbytes = stag_vector_bytes(ctx, prec);
    const size_t vec_sz = align256(vbytes);
    char *s = static_cast<char *>(dev_scratch);
    double *canon = reinterpret_cast<double *>(s);
    char *b = s + canon_sz, *y = b + vec_sz, *x = y + vec_sz;
    // x_i are contiguous at stride stag_vector_bytes (ABI of stag_mshift_cg); round the block up
    char *ws = x + align256((size_t)nshift * vbytes);
    STAG_CUDA_OK(cudaMemcpyAsync(canon, host_b, cbytes, cudaMemcpyHostToDevice, st));
    int rc = stag_vector_pack(ctx, canon, b, prec, st);
    if (rc) return rc;
    const int cg_rc = stag_mshift_cg(ctx, packed, prec, recon, b, mass, nshift, host_shifts,
                                     host_residues, residue0, stop, maxiter, x,
                                     host_y ? y : nullptr, ws, info, st);
    if (cg_rc != STAG_OK && cg_rc != STAG_ERR_NOTCONV && cg_rc != STAG_ERR_BREAKDOWN) return cg_rc;
    for (int i = 0; i < nshift; ++i) {
        rc = stag_vector_unpack(ctx, x + (size_t)i * vbytes, prec, canon, st);
        if (rc) return rc;
        STAG_CUDA_OK(cudaMemcpyAsync(host_x + (size_t)i * (cbytes / sizeof(double)), canon, cbytes,
                                     cudaMemcpyDeviceToHost, st));
    }
    if (host_y) {
        rc = stag_vector_unpack(ctx, y, prec, canon, st);
        if (rc) return rc;
        STAG_CUDA_OK(cudaMemcpyAsync(host_y, canon, cbytes, cudaMemcpyDeviceToHost, st));
    }
    STAG_CUDA_OK(cudaStreamSynchronize(st));
    return cg_rc;
}
