// launch.h - internal host-side launchers (one per kernel family).  The C ABI in api.cu validates
// arguments and calls these; nothing here is exported.
//
// Every kernel family takes a BATCH of jobs by value (kernel parameters): block (x, y) works on job y.  The
// single-buffer entry points launch a batch of one; the ring engine (ring.cu) launches one batch per kernel
// family per ring step with one job per logical rank (SURVEY.md S7 hard part 5, S8(b) "batched form").
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace pici {

// A job runs only if its gate is open: ptr == nullptr, or (*ptr & mask) == value when the kernel starts
// (include/pici.h "Gating").
struct Gate {
    const int32_t *ptr;
    int32_t mask;
    int32_t value;
};
inline Gate gate_eq(const int32_t *p, int32_t v) { return Gate{p, -1, v}; }
constexpr int kMaxBatch = 16;

int num_sms();  // cached cudaDevAttrMultiProcessorCount of the current device

// Index (0..63) of the current device: one-time per-kernel setup (cudaFuncSetAttribute, occupancy) is kept
// per device, so a process that drives several GPUs configures each of them.
inline int current_device_slot() {
    int dev = 0;
    cudaGetDevice(&dev);
    return (dev < 0 || dev >= 64) ? 0 : dev;
}

uint64_t scan_workspace_bytes(uint64_t n);

struct CompressJob {
    const void *dense;
    uint64_t n;
    uint64_t *B;
    uint32_t *I;
    void *A;
    void *ws;
    Gate gate;
    // prune-and-compress (pici_prune_compress, include/pici_prune.h): `dense` is the gradient g, resid the error-
    // feedback buffer e (updated in place), *d_tau the magnitude threshold; unused (nullptr) by plain compress
    float *resid;
    const float *d_tau;
    float leak;
};
cudaError_t launch_compress_batch(const CompressJob *jobs, int count, int dtype, cudaStream_t s);
cudaError_t launch_prune_compress(const CompressJob &job, cudaStream_t s);   // fp32, one job
cudaError_t launch_compress(const void *dense, uint64_t n, int dtype, uint64_t *B, uint32_t *I, void *A,
                            void *ws, Gate g, cudaStream_t s);

// mode 0: decompress (overwrite), 1: out = local + sparse (reduce_sd, out may alias local).
// d_switch / nnz_switch: if d_switch != nullptr the kernel first evaluates switched = I[T] >= nnz_switch,
// writes *d_switch = switched ? on_value : off_value and does nothing else unless switched.
struct DensifyCtl {
    int32_t *d_flag;      // nullptr = unconditional
    uint64_t nnz_switch;
    int32_t on_value, off_value;
};
struct ExpandJob {
    const uint64_t *B;
    const uint32_t *I;
    const void *A;
    uint64_t n;
    const void *local;
    void *out;
    DensifyCtl ctl;
    Gate gate;
};
cudaError_t launch_expand_batch(const ExpandJob *jobs, int count, int dtype, int mode, cudaStream_t s);
cudaError_t launch_expand(const uint64_t *B, const uint32_t *I, const void *A, uint64_t n, int dtype,
                          const void *local, void *out, int mode, DensifyCtl ctl, Gate g, cudaStream_t s);

struct MergeJob {
    const uint64_t *Bx;
    const uint32_t *Ix;
    const void *Ax;
    const uint64_t *By;
    const uint32_t *Iy;
    const void *Ay;
    uint64_t n;
    uint64_t *Bo;
    uint32_t *Io;
    void *Ao;
    void *ws;
    Gate gate;
};
cudaError_t launch_reduce_ss_batch(const MergeJob *jobs, int count, cudaStream_t s);
cudaError_t launch_reduce_ss(const uint64_t *Bx, const uint32_t *Ix, const void *Ax, const uint64_t *By,
                             const uint32_t *Iy, const void *Ay, uint64_t n, uint64_t *Bo, uint32_t *Io,
                             void *Ao, void *ws, Gate g, cudaStream_t s);

cudaError_t launch_nnz_pici(const uint32_t *I, uint64_t n, uint32_t *d_nnz, cudaStream_t s);
cudaError_t launch_nnz_dense(const void *dense, uint64_t n, int dtype, uint32_t *d_nnz, cudaStream_t s);

struct DenseAddJob {
    const void *recv;
    const void *local;
    uint64_t n;
    void *out;
    int32_t *d_fmt_out;
    Gate gate;
};
cudaError_t launch_dense_add_batch(const DenseAddJob *jobs, int count, cudaStream_t s);
cudaError_t launch_dense_add_bf16(const void *recv, const void *local, uint64_t n, void *out, int32_t *d_fmt_out, Gate g,
                                  cudaStream_t s);
cudaError_t launch_dense_add(const void *recv, const void *local, uint64_t n, void *out, int32_t *d_fmt_out,
                             Gate g, cudaStream_t s);

struct DenseCopyJob {
    const void *src;
    void *dst;
    uint64_t nbytes;
    Gate gate;
};
cudaError_t launch_dense_copy_batch(const DenseCopyJob *jobs, int count, cudaStream_t s);
cudaError_t launch_dense_copy(const void *src, void *dst, uint64_t nbytes, Gate g, cudaStream_t s);
cudaError_t launch_set_u32(uint32_t *p, uint32_t v, Gate g, cudaStream_t s);
cudaError_t launch_probe_rmw(const uint32_t *idx, uint64_t m, void *dense, cudaStream_t s);

template <class Job>
struct Batch {
    Job job[kMaxBatch];
};

}  // namespace pici
