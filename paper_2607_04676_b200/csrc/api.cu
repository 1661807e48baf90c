// api.cu - the C ABI of libpici_b200 (include/pici.h): host-side argument validation, then one or two
// kernel launches on the caller's stream.  No allocation, no global state besides cached device
// attributes, no synchronisation except in the *_host forms.
#include "../../include/pici.h"
#include "launch.h"
#include "pici_common.cuh"

using namespace pici;

namespace {

inline bool aligned(const void *p, uintptr_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) == 0; }
inline bool bad_dtype(int dt) { return dt != PICI_F32 && dt != PICI_BF16; }
inline uint64_t tiles(uint64_t n) { return (n + kTile - 1) / kTile; }
inline size_t esize(int dt) { return dt == PICI_F32 ? 4 : 2; }
inline int cuda_rc(cudaError_t e) { return e == cudaSuccess ? PICI_OK : PICI_ERR_CUDA; }
constexpr uint64_t kMaxN = 1ull << 32;
const Gate kOpen = {nullptr, 0, 0};

int check_pici(const uint64_t *B, const uint32_t *I, const void *A, uint64_t n, int dtype) {
    if (bad_dtype(dtype)) return PICI_ERR_DTYPE;
    if (n >= kMaxN || I == nullptr) return PICI_ERR_INVALID_ARG;
    if (n != 0 && (B == nullptr || A == nullptr)) return PICI_ERR_INVALID_ARG;
    if (!aligned(B, 16) || !aligned(A, 16) || !aligned(I, 4)) return PICI_ERR_ALIGN;
    return PICI_OK;
}

int do_compress(const void *dense, uint64_t n, int dtype, uint64_t *B, uint32_t *I, void *A, uint64_t A_capacity,
                void *ws, uint64_t ws_bytes, Gate g, void *stream) {
    int rc = check_pici(B, I, A, n, dtype);
    if (rc != PICI_OK) return rc;
    if (n != 0 && dense == nullptr) return PICI_ERR_INVALID_ARG;
    if (!aligned(dense, 16) || !aligned(ws, 16)) return PICI_ERR_ALIGN;
    if (A_capacity < n) return PICI_ERR_CAPACITY;
    if (n != 0 && (ws == nullptr || ws_bytes < scan_workspace_bytes(n))) return PICI_ERR_WORKSPACE;
    return cuda_rc(launch_compress(dense, n, dtype, B, I, A, ws, g, static_cast<cudaStream_t>(stream)));
}

int do_expand(const uint64_t *B, const uint32_t *I, const void *A, uint64_t n, int dtype, const void *local,
              void *out, int mode, DensifyCtl ctl, Gate g, void *stream) {
    int rc = check_pici(B, I, A, n, dtype);
    if (rc != PICI_OK) return rc;
    if (n != 0 && out == nullptr && ctl.d_flag == nullptr) return PICI_ERR_INVALID_ARG;
    if (n != 0 && mode == 1 && local == nullptr) return PICI_ERR_INVALID_ARG;
    if (!aligned(out, 16) || !aligned(local, 16)) return PICI_ERR_ALIGN;
    return cuda_rc(launch_expand(B, I, A, n, dtype, local, out, mode, ctl, g, static_cast<cudaStream_t>(stream)));
}

int do_reduce_ss(const uint64_t *Bx, const uint32_t *Ix, const void *Ax, const uint64_t *By, const uint32_t *Iy,
                 const void *Ay, uint64_t n, int dtype, uint64_t *Bo, uint32_t *Io, void *Ao, uint64_t Ao_capacity,
                 void *ws, uint64_t ws_bytes, Gate g, void *stream) {
    if (bad_dtype(dtype)) return PICI_ERR_DTYPE;
    if (dtype != PICI_F32) return PICI_ERR_DTYPE;
    int rc = check_pici(Bx, Ix, Ax, n, dtype);
    if (rc == PICI_OK) rc = check_pici(By, Iy, Ay, n, dtype);
    if (rc == PICI_OK) rc = check_pici(Bo, Io, Ao, n, dtype);
    if (rc != PICI_OK) return rc;
    if (!aligned(ws, 16)) return PICI_ERR_ALIGN;
    if (Ao_capacity < n) return PICI_ERR_CAPACITY;
    if (n != 0 && (ws == nullptr || ws_bytes < scan_workspace_bytes(n))) return PICI_ERR_WORKSPACE;
    // "Outputs must not alias inputs": the merge reads X and Y while it writes O
    if (n != 0 && (Bo == Bx || Bo == By || Io == Ix || Io == Iy || Ao == Ax || Ao == Ay)) return PICI_ERR_INVALID_ARG;
    return cuda_rc(launch_reduce_ss(Bx, Ix, Ax, By, Iy, Ay, n, Bo, Io, Ao, ws, g, static_cast<cudaStream_t>(stream)));
}

}  // namespace

extern "C" {

int pici_version(void) { return PICI_VERSION; }

const char *pici_strerror(int code) {
    switch (code) {
        case PICI_OK: return "ok";
        case PICI_ERR_INVALID_ARG: return "invalid argument (null pointer, n >= 2^32 or bad flag)";
        case PICI_ERR_DTYPE: return "unknown dtype or dtype not supported by this call";
        case PICI_ERR_ALIGN: return "pointer alignment violated";
        case PICI_ERR_CAPACITY: return "values capacity smaller than n";
        case PICI_ERR_WORKSPACE: return "workspace too small";
        case PICI_ERR_CUDA: return "CUDA runtime or launch failure";
        default: return "unknown error code";
    }
}

int pici_sizes(uint64_t n, int dtype, uint64_t *bitvec_words, uint64_t *index_entries, uint64_t *values_capacity,
               uint64_t *workspace_bytes) {
    if (bad_dtype(dtype)) return PICI_ERR_DTYPE;
    if (n >= kMaxN) return PICI_ERR_INVALID_ARG;
    const uint64_t T = tiles(n);
    if (bitvec_words) *bitvec_words = 64 * T;
    if (index_entries) *index_entries = T + 1;
    if (values_capacity) *values_capacity = n;
    if (workspace_bytes) *workspace_bytes = scan_workspace_bytes(n);
    return PICI_OK;
}

int pici_workspace_init(void *ws, uint64_t ws_bytes, void *stream) {
    if (ws == nullptr) return ws_bytes == 0 ? PICI_OK : PICI_ERR_INVALID_ARG;
    if (!aligned(ws, 16)) return PICI_ERR_ALIGN;
    if (ws_bytes == 0) return PICI_OK;
    return cuda_rc(cudaMemsetAsync(ws, 0, ws_bytes, static_cast<cudaStream_t>(stream)));
}

int pici_compress(const void *dense, uint64_t n, int dtype, uint64_t *B, uint32_t *I, void *A, uint64_t A_capacity,
                  void *ws, uint64_t ws_bytes, void *stream) {
    return do_compress(dense, n, dtype, B, I, A, A_capacity, ws, ws_bytes, kOpen, stream);
}

int pici_compress_gated(const void *dense, uint64_t n, int dtype, uint64_t *B, uint32_t *I, void *A,
                        uint64_t A_capacity, void *ws, uint64_t ws_bytes, const int32_t *d_gate, int32_t gate_value,
                        void *stream) {
    return do_compress(dense, n, dtype, B, I, A, A_capacity, ws, ws_bytes, gate_eq(d_gate, gate_value), stream);
}

int pici_decompress(const uint64_t *B, const uint32_t *I, const void *A, uint64_t n, int dtype, void *dense_out,
                    void *stream) {
    return do_expand(B, I, A, n, dtype, nullptr, dense_out, 0, DensifyCtl{nullptr, 0, 0, 0}, kOpen, stream);
}

int pici_decompress_gated(const uint64_t *B, const uint32_t *I, const void *A, uint64_t n, int dtype, void *dense_out,
                          const int32_t *d_gate, int32_t gate_value, void *stream) {
    return do_expand(B, I, A, n, dtype, nullptr, dense_out, 0, DensifyCtl{nullptr, 0, 0, 0}, gate_eq(d_gate, gate_value),
                     stream);
}

int pici_reduce_sd(const uint64_t *B, const uint32_t *I, const void *A, uint64_t n, int dtype, void *dense_inout,
                   void *stream) {
    return do_expand(B, I, A, n, dtype, dense_inout, dense_inout, 1, DensifyCtl{nullptr, 0, 0, 0}, kOpen, stream);
}

int pici_reduce_sd_out_gated(const uint64_t *B, const uint32_t *I, const void *A, const void *local, uint64_t n,
                             int dtype, void *out, const int32_t *d_gate, int32_t gate_value, void *stream) {
    return do_expand(B, I, A, n, dtype, local, out, 1, DensifyCtl{nullptr, 0, 0, 0}, gate_eq(d_gate, gate_value), stream);
}

int pici_reduce_ss(const uint64_t *Bx, const uint32_t *Ix, const void *Ax, const uint64_t *By, const uint32_t *Iy,
                   const void *Ay, uint64_t n, int dtype, uint64_t *Bo, uint32_t *Io, void *Ao, uint64_t Ao_capacity,
                   void *ws, uint64_t ws_bytes, void *stream) {
    return do_reduce_ss(Bx, Ix, Ax, By, Iy, Ay, n, dtype, Bo, Io, Ao, Ao_capacity, ws, ws_bytes, kOpen, stream);
}

int pici_reduce_ss_gated(const uint64_t *Bx, const uint32_t *Ix, const void *Ax, const uint64_t *By,
                         const uint32_t *Iy, const void *Ay, uint64_t n, int dtype, uint64_t *Bo, uint32_t *Io,
                         void *Ao, uint64_t Ao_capacity, void *ws, uint64_t ws_bytes, const int32_t *d_gate,
                         int32_t gate_value, void *stream) {
    return do_reduce_ss(Bx, Ix, Ax, By, Iy, Ay, n, dtype, Bo, Io, Ao, Ao_capacity, ws, ws_bytes,
                        gate_eq(d_gate, gate_value), stream);
}

int pici_nnz(const uint32_t *I, uint64_t n, uint32_t *d_nnz, void *stream) {
    if (I == nullptr || d_nnz == nullptr || n >= kMaxN) return PICI_ERR_INVALID_ARG;
    if (!aligned(I, 4) || !aligned(d_nnz, 4)) return PICI_ERR_ALIGN;
    return cuda_rc(launch_nnz_pici(I, n, d_nnz, static_cast<cudaStream_t>(stream)));
}

int pici_nnz_dense(const void *dense, uint64_t n, int dtype, uint32_t *d_nnz, void *ws, uint64_t ws_bytes,
                   void *stream) {
    (void)ws;
    (void)ws_bytes;
    if (bad_dtype(dtype)) return PICI_ERR_DTYPE;
    if (d_nnz == nullptr || n >= kMaxN || (n != 0 && dense == nullptr)) return PICI_ERR_INVALID_ARG;
    if (!aligned(dense, 16) || !aligned(d_nnz, 4)) return PICI_ERR_ALIGN;
    return cuda_rc(launch_nnz_dense(dense, n, dtype, d_nnz, static_cast<cudaStream_t>(stream)));
}

int pici_maybe_densify(const uint64_t *B, const uint32_t *I, const void *A, uint64_t n, int dtype,
                       uint64_t nnz_switch, void *dense_out, int32_t *d_switched, void *stream) {
    if (d_switched == nullptr) return PICI_ERR_INVALID_ARG;
    return do_expand(B, I, A, n, dtype, nullptr, dense_out, 0, DensifyCtl{d_switched, nnz_switch, 1, 0}, kOpen, stream);
}

int pici_maybe_densify_gated(const uint64_t *B, const uint32_t *I, const void *A, uint64_t n, int dtype,
                             uint64_t nnz_switch, void *dense_out, int32_t *d_fmt_out, const int32_t *d_gate,
                             int32_t gate_value, void *stream) {
    if (d_fmt_out == nullptr || d_fmt_out == d_gate) return PICI_ERR_INVALID_ARG;
    return do_expand(B, I, A, n, dtype, nullptr, dense_out, 0,
                     DensifyCtl{d_fmt_out, nnz_switch, PICI_FMT_DENSE, PICI_FMT_PICI}, gate_eq(d_gate, gate_value), stream);
}

int pici_dense_add_gated(const void *recv, const void *local, uint64_t n, int dtype, void *out, int32_t *d_fmt_out,
                         const int32_t *d_gate, int32_t gate_value, void *stream) {
    if (bad_dtype(dtype)) return PICI_ERR_DTYPE;
    if (n >= kMaxN || (n != 0 && (recv == nullptr || local == nullptr || out == nullptr))) return PICI_ERR_INVALID_ARG;
    if (d_fmt_out != nullptr && d_fmt_out == d_gate) return PICI_ERR_INVALID_ARG;
    if (!aligned(recv, 16) || !aligned(local, 16) || !aligned(out, 16)) return PICI_ERR_ALIGN;
    return cuda_rc((dtype == PICI_F32 ? launch_dense_add : launch_dense_add_bf16)(recv, local, n, out, d_fmt_out,
                                                                                 gate_eq(d_gate, gate_value),
                                                                                 static_cast<cudaStream_t>(stream)));
}

int pici_dense_copy_gated(const void *src, void *dst, uint64_t n, int dtype, const int32_t *d_gate, int32_t gate_value,
                          void *stream) {
    if (bad_dtype(dtype)) return PICI_ERR_DTYPE;
    if (n >= kMaxN || (n != 0 && (src == nullptr || dst == nullptr))) return PICI_ERR_INVALID_ARG;
    if (!aligned(src, 16) || !aligned(dst, 16)) return PICI_ERR_ALIGN;
    if (n == 0) return PICI_OK;
    return cuda_rc(launch_dense_copy(src, dst, n * esize(dtype), gate_eq(d_gate, gate_value), static_cast<cudaStream_t>(stream)));
}

int pici_probe_random_rmw(const uint32_t *d_idx, uint64_t m, void *dense_inout, uint64_t n, void *stream) {
    if (m != 0 && (d_idx == nullptr || dense_inout == nullptr)) return PICI_ERR_INVALID_ARG;
    if (n >= kMaxN) return PICI_ERR_INVALID_ARG;
    if (!aligned(d_idx, 4) || !aligned(dense_inout, 16)) return PICI_ERR_ALIGN;
    return cuda_rc(launch_probe_rmw(d_idx, m, dense_inout, static_cast<cudaStream_t>(stream)));
}

int pici_compress_host(const void *h_dense, uint64_t n, int dtype, uint64_t *h_B, uint32_t *h_I, void *h_A,
                       uint64_t *h_nnz, void *d_dense, uint64_t *d_B, uint32_t *d_I, void *d_A, void *ws,
                       uint64_t ws_bytes, void *stream) {
    if (bad_dtype(dtype)) return PICI_ERR_DTYPE;
    if (h_I == nullptr || h_nnz == nullptr || (n != 0 && (h_dense == nullptr || h_B == nullptr || h_A == nullptr)))
        return PICI_ERR_INVALID_ARG;
    if (n >= kMaxN || d_I == nullptr || (n != 0 && (d_dense == nullptr || d_B == nullptr || d_A == nullptr))) return PICI_ERR_INVALID_ARG;
    if (!aligned(d_dense, 16) || !aligned(d_B, 16) || !aligned(d_A, 16) || !aligned(d_I, 4) || !aligned(ws, 16)) return PICI_ERR_ALIGN;
    if (n != 0 && (ws == nullptr || ws_bytes < scan_workspace_bytes(n))) return PICI_ERR_WORKSPACE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const uint64_t T = tiles(n);
    if (n != 0 && cudaMemcpyAsync(d_dense, h_dense, n * esize(dtype), cudaMemcpyHostToDevice, s) != cudaSuccess)
        return PICI_ERR_CUDA;
    int rc = pici_compress(d_dense, n, dtype, d_B, d_I, d_A, n, ws, ws_bytes, stream);
    if (rc != PICI_OK) return rc;
    if (cudaMemcpyAsync(h_I, d_I, (T + 1) * sizeof(uint32_t), cudaMemcpyDeviceToHost, s) != cudaSuccess) return PICI_ERR_CUDA;
    if (n != 0 && cudaMemcpyAsync(h_B, d_B, 64 * T * sizeof(uint64_t), cudaMemcpyDeviceToHost, s) != cudaSuccess)
        return PICI_ERR_CUDA;
    if (cudaStreamSynchronize(s) != cudaSuccess) return PICI_ERR_CUDA;
    const uint64_t nnz = h_I[T];
    *h_nnz = nnz;
    if (nnz != 0) {
        if (cudaMemcpyAsync(h_A, d_A, nnz * esize(dtype), cudaMemcpyDeviceToHost, s) != cudaSuccess) return PICI_ERR_CUDA;
        if (cudaStreamSynchronize(s) != cudaSuccess) return PICI_ERR_CUDA;
    }
    return PICI_OK;
}

int pici_decompress_host(const uint64_t *h_B, const uint32_t *h_I, const void *h_A, uint64_t nnz, uint64_t n,
                         int dtype, void *h_dense_out, uint64_t *d_B, uint32_t *d_I, void *d_A, void *d_dense,
                         void *stream) {
    if (bad_dtype(dtype)) return PICI_ERR_DTYPE;
    if (h_I == nullptr || nnz > n || (n != 0 && (h_B == nullptr || h_dense_out == nullptr)) || (nnz != 0 && h_A == nullptr))
        return PICI_ERR_INVALID_ARG;
    if (n >= kMaxN || d_I == nullptr || (n != 0 && (d_dense == nullptr || d_B == nullptr || d_A == nullptr))) return PICI_ERR_INVALID_ARG;
    if (!aligned(d_dense, 16) || !aligned(d_B, 16) || !aligned(d_A, 16) || !aligned(d_I, 4)) return PICI_ERR_ALIGN;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const uint64_t T = tiles(n);
    if (cudaMemcpyAsync(d_I, h_I, (T + 1) * sizeof(uint32_t), cudaMemcpyHostToDevice, s) != cudaSuccess) return PICI_ERR_CUDA;
    if (n != 0 && cudaMemcpyAsync(d_B, h_B, 64 * T * sizeof(uint64_t), cudaMemcpyHostToDevice, s) != cudaSuccess)
        return PICI_ERR_CUDA;
    if (nnz != 0 && cudaMemcpyAsync(d_A, h_A, nnz * esize(dtype), cudaMemcpyHostToDevice, s) != cudaSuccess)
        return PICI_ERR_CUDA;
    int rc = pici_decompress(d_B, d_I, d_A, n, dtype, d_dense, stream);
    if (rc != PICI_OK) return rc;
    if (n != 0 && cudaMemcpyAsync(h_dense_out, d_dense, n * esize(dtype), cudaMemcpyDeviceToHost, s) != cudaSuccess)
        return PICI_ERR_CUDA;
    return cuda_rc(cudaStreamSynchronize(s));
}

}  // extern "C"
