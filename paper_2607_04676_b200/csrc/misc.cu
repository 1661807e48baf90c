// misc.cu - the small kernels of the path: pici_nnz, pici_nnz_dense (the on-device
// measurement the paper lacks after a scatter-add), the dense+dense ring step (the
// paper's reduceCopy) and a gated 32-bit store.
#include "launch.h"
#include "pici_common.cuh"
#include "../../include/pici.h"

namespace pici {

// The streaming kernels below are grid-stride loops.  A grid of exactly one resident wave gives every SM the same
// share and the launch ends with the slowest SM (a 16-byte-store fill of 1 GiB: 6.0 TB/s with 1184 CTAs, 7.2 TB/s with
// 65536); several waves of CTAs let the block scheduler balance them.  Single ungated launches only: the ring engine's
// batched, gated launches (half of which return at once) pay for every extra CTA.
constexpr uint64_t kStreamWaves = 16;

__global__ void set_u32_kernel(uint32_t *p, uint32_t v, Gate gate) {
    if (gate_closed(gate.ptr, gate.mask, gate.value)) return;
    *p = v;
}

cudaError_t launch_set_u32(uint32_t *p, uint32_t v, Gate g, cudaStream_t s) {
    set_u32_kernel<<<1, 1, 0, s>>>(p, v, g);
    return cudaGetLastError();
}

__global__ void nnz_pici_kernel(const uint32_t *__restrict__ I, uint32_t T, uint32_t *d_nnz) { *d_nnz = I[T]; }

cudaError_t launch_nnz_pici(const uint32_t *I, uint64_t n, uint32_t *d_nnz, cudaStream_t s) {
    nnz_pici_kernel<<<1, 1, 0, s>>>(I, (uint32_t)((n + kTile - 1) / kTile), d_nnz);
    return cudaGetLastError();
}

// Count of nz(x) over a dense buffer.  128-bit loads, 4 in flight per thread; integer atomics, so the
// result does not depend on scheduling.
template <int DT>
__global__ void __launch_bounds__(256) nnz_dense_kernel(const void *__restrict__ dense, uint64_t n, uint32_t *d_nnz) {
    constexpr int kPerVec = DT == PICI_F32 ? 4 : 8;
    const uint64_t nvec = n / kPerVec;
    const uint4 *p = reinterpret_cast<const uint4 *>(dense);
    uint32_t cnt = 0;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    auto count4 = [&](uint4 v) {
        if constexpr (DT == PICI_F32) {
            cnt += nz32(v.x) + nz32(v.y) + nz32(v.z) + nz32(v.w);
        } else {
            cnt += nz16lo(v.x) + nz16hi(v.x) + nz16lo(v.y) + nz16hi(v.y) + nz16lo(v.z) + nz16hi(v.z) + nz16lo(v.w) + nz16hi(v.w);
        }
    };
    for (; i + 3 * stride < nvec; i += 4 * stride) {
        uint4 a = ldg_nc_u4(p + i), b = ldg_nc_u4(p + i + stride), c = ldg_nc_u4(p + i + 2 * stride), d = ldg_nc_u4(p + i + 3 * stride);
        count4(a); count4(b); count4(c); count4(d);
    }
    for (; i < nvec; i += stride) count4(ldg_nc_u4(p + i));
    if (blockIdx.x == 0 && threadIdx.x == 0) {  // ragged tail (< one vector)
        for (uint64_t j = nvec * kPerVec; j < n; ++j) {
            if constexpr (DT == PICI_F32) cnt += nz32(reinterpret_cast<const uint32_t *>(dense)[j]);
            else cnt += nz16lo(reinterpret_cast<const uint16_t *>(dense)[j]);
        }
    }
    cnt = warp_sum(cnt);
    __shared__ uint32_t part[8];
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = cnt;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t s = 0;
        for (int w = 0; w < 8; ++w) s += part[w];
        if (s) atomicAdd(d_nnz, s);
    }
}

cudaError_t launch_nnz_dense(const void *dense, uint64_t n, int dtype, uint32_t *d_nnz, cudaStream_t s) {
    cudaError_t e = cudaMemsetAsync(d_nnz, 0, sizeof(uint32_t), s);
    if (e != cudaSuccess || n == 0) return e;
    const uint64_t nvec = n / (dtype == PICI_F32 ? 4 : 8);
    uint64_t blocks = (nvec + 256 * 4 - 1) / (256 * 4);
    const uint64_t cap = (uint64_t)num_sms() * 8 * kStreamWaves;
    if (blocks > cap) blocks = cap;
    if (blocks == 0) blocks = 1;
    if (dtype == PICI_F32) nnz_dense_kernel<PICI_F32><<<(unsigned)blocks, 256, 0, s>>>(dense, n, d_nnz);
    else nnz_dense_kernel<PICI_BF16><<<(unsigned)blocks, 256, 0, s>>>(dense, n, d_nnz);
    return cudaGetLastError();
}

// out[i] = recv[i] + local[i], one fp32 add each, order "received + local" (C9 #7).
__global__ void __launch_bounds__(256) dense_add_kernel(const Batch<DenseAddJob> batch) {
    const DenseAddJob &job = batch.job[blockIdx.y];
    if (gate_closed(job.gate.ptr, job.gate.mask, job.gate.value)) return;
    const float *recv = reinterpret_cast<const float *>(job.recv), *local = reinterpret_cast<const float *>(job.local);
    float *out = reinterpret_cast<float *>(job.out);
    const uint64_t n = job.n;
    int32_t *d_fmt_out = job.d_fmt_out;
    if (d_fmt_out != nullptr && blockIdx.x == 0 && threadIdx.x == 0) *d_fmt_out = PICI_FMT_DENSE;
    const uint64_t nvec = n / 4;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const uint4 *a = reinterpret_cast<const uint4 *>(recv), *b = reinterpret_cast<const uint4 *>(local);
    uint4 *o = reinterpret_cast<uint4 *>(out);
    auto add4 = [](uint4 x, uint4 y) {
        uint4 r;
        r.x = __float_as_uint(__fadd_rn(__uint_as_float(x.x), __uint_as_float(y.x)));
        r.y = __float_as_uint(__fadd_rn(__uint_as_float(x.y), __uint_as_float(y.y)));
        r.z = __float_as_uint(__fadd_rn(__uint_as_float(x.z), __uint_as_float(y.z)));
        r.w = __float_as_uint(__fadd_rn(__uint_as_float(x.w), __uint_as_float(y.w)));
        return r;
    };
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + stride < nvec; i += 2 * stride) {
        uint4 x0 = ldg_stream_u4(a + i), y0 = ldg_stream_u4(b + i);
        uint4 x1 = ldg_stream_u4(a + i + stride), y1 = ldg_stream_u4(b + i + stride);
        stg_stream_u4(o + i, add4(x0, y0));
        stg_stream_u4(o + i + stride, add4(x1, y1));
    }
    for (; i < nvec; i += stride) stg_stream_u4(o + i, add4(ldg_stream_u4(a + i), ldg_stream_u4(b + i)));
    if (blockIdx.x == 0 && threadIdx.x == 0)
        for (uint64_t j = nvec * 4; j < n; ++j) out[j] = __fadd_rn(recv[j], local[j]);
}

cudaError_t launch_dense_add_batch(const DenseAddJob *jobs, int count, cudaStream_t s) {
    if (count <= 0) return cudaSuccess;
    if (count > kMaxBatch) return cudaErrorInvalidValue;
    Batch<DenseAddJob> batch;
    uint64_t nvec = 0;
    for (int j = 0; j < count; ++j) {
        batch.job[j] = jobs[j];
        nvec = max(nvec, jobs[j].n / 4);
    }
    uint64_t blocks = (nvec + 256 * 2 - 1) / (256 * 2);
    const uint64_t waves = (count == 1 && jobs[0].gate.ptr == nullptr) ? kStreamWaves : 1;   // see kStreamWaves
    const uint64_t cap = max((uint64_t)num_sms() * 8 * waves / count, (uint64_t)1);
    if (blocks > cap) blocks = cap;
    if (blocks == 0) blocks = 1;
    dense_add_kernel<<<dim3((unsigned)blocks, (unsigned)count), 256, 0, s>>>(batch);
    return cudaGetLastError();
}

cudaError_t launch_dense_add(const void *recv, const void *local, uint64_t n, void *out, int32_t *d_fmt_out, Gate g,
                             cudaStream_t s) {
    const DenseAddJob job = {recv, local, n, out, d_fmt_out, g};
    return launch_dense_add_batch(&job, 1, s);
}

// bf16: out[i] = bf16(recv[i] + local[i]) - widened to fp32, one fp32 add, rounded to nearest even (pici_common.cuh).
__global__ void __launch_bounds__(256) dense_add_bf16_kernel(const DenseAddJob job) {
    if (gate_closed(job.gate.ptr, job.gate.mask, job.gate.value)) return;
    const uint16_t *recv = reinterpret_cast<const uint16_t *>(job.recv), *local = reinterpret_cast<const uint16_t *>(job.local);
    uint16_t *out = reinterpret_cast<uint16_t *>(job.out);
    const uint64_t n = job.n;
    if (job.d_fmt_out != nullptr && blockIdx.x == 0 && threadIdx.x == 0) *job.d_fmt_out = PICI_FMT_DENSE;
    const uint64_t nvec = n / 8;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const uint4 *a = reinterpret_cast<const uint4 *>(recv), *b = reinterpret_cast<const uint4 *>(local);
    uint4 *o = reinterpret_cast<uint4 *>(out);
    auto add2 = [](uint32_t x, uint32_t y) {
        return bf16_add_bits(x & 0xFFFFu, y & 0xFFFFu) | (bf16_add_bits(x >> 16, y >> 16) << 16);
    };
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += stride) {
        const uint4 x = ldg_stream_u4(a + i), y = ldg_stream_u4(b + i);
        stg_stream_u4(o + i, make_uint4(add2(x.x, y.x), add2(x.y, y.y), add2(x.z, y.z), add2(x.w, y.w)));
    }
    if (blockIdx.x == 0 && threadIdx.x == 0)
        for (uint64_t j = nvec * 8; j < n; ++j) out[j] = (uint16_t)bf16_add_bits(recv[j], local[j]);
}

cudaError_t launch_dense_add_bf16(const void *recv, const void *local, uint64_t n, void *out, int32_t *d_fmt_out, Gate g,
                                  cudaStream_t s) {
    const DenseAddJob job = {recv, local, n, out, d_fmt_out, g};
    uint64_t blocks = (n / 8 + 255) / 256;
    const uint64_t cap = (uint64_t)num_sms() * 8 * (g.ptr == nullptr ? kStreamWaves : 1);
    if (blocks > cap) blocks = cap;
    if (blocks == 0) blocks = 1;
    dense_add_bf16_kernel<<<(unsigned)blocks, 256, 0, s>>>(job);
    return cudaGetLastError();
}

// dst[i] = src[i] (bit copy), gated: a dense message landing in its all-gather slot.
__global__ void __launch_bounds__(256) dense_copy_kernel(const Batch<DenseCopyJob> batch) {
    const DenseCopyJob &job = batch.job[blockIdx.y];
    if (gate_closed(job.gate.ptr, job.gate.mask, job.gate.value)) return;
    const uint4 *src = reinterpret_cast<const uint4 *>(job.src);
    uint4 *dst = reinterpret_cast<uint4 *>(job.dst);
    const uint64_t nbytes = job.nbytes;
    const uint64_t nvec = nbytes / 16;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + 3 * stride < nvec; i += 4 * stride) {
        uint4 a = ldg_stream_u4(src + i), b = ldg_stream_u4(src + i + stride), c = ldg_stream_u4(src + i + 2 * stride),
              d = ldg_stream_u4(src + i + 3 * stride);
        stg_stream_u4(dst + i, a);
        stg_stream_u4(dst + i + stride, b);
        stg_stream_u4(dst + i + 2 * stride, c);
        stg_stream_u4(dst + i + 3 * stride, d);
    }
    for (; i < nvec; i += stride) stg_stream_u4(dst + i, ldg_stream_u4(src + i));
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        const unsigned char *s8 = reinterpret_cast<const unsigned char *>(src);
        unsigned char *d8 = reinterpret_cast<unsigned char *>(dst);
        for (uint64_t j = nvec * 16; j < nbytes; ++j) d8[j] = s8[j];
    }
}

cudaError_t launch_dense_copy_batch(const DenseCopyJob *jobs, int count, cudaStream_t s) {
    if (count <= 0) return cudaSuccess;
    if (count > kMaxBatch) return cudaErrorInvalidValue;
    Batch<DenseCopyJob> batch;
    uint64_t nvec = 0;
    for (int j = 0; j < count; ++j) {
        batch.job[j] = jobs[j];
        nvec = max(nvec, jobs[j].nbytes / 16);
    }
    uint64_t blocks = (nvec + 256 * 4 - 1) / (256 * 4);
    const uint64_t waves = (count == 1 && jobs[0].gate.ptr == nullptr) ? kStreamWaves : 1;
    const uint64_t cap = max((uint64_t)num_sms() * 8 * waves / count, (uint64_t)1);
    if (blocks > cap) blocks = cap;
    if (blocks == 0) blocks = 1;
    dense_copy_kernel<<<dim3((unsigned)blocks, (unsigned)count), 256, 0, s>>>(batch);
    return cudaGetLastError();
}

cudaError_t launch_dense_copy(const void *src, void *dst, uint64_t nbytes, Gate g, cudaStream_t s) {
    const DenseCopyJob job = {src, dst, nbytes, g};
    return launch_dense_copy_batch(&job, 1, s);
}

// ---- measurement aid: the bare random read-modify-write stream (include/pici.h pici_probe_random_rmw) -------------
// dense[idx[i]] = dense[idx[i]] + 1.0f for i < m, one thread per index, the gather through the same
// ld.global.L2::64B instruction reduce_sd's sparse regime uses, nothing else: what the memory system gives for
// this access pattern, against which bench.py reports reduce_sd's read-modify-write regime.
__global__ void __launch_bounds__(256) probe_rmw_kernel(const uint32_t *__restrict__ idx, uint64_t m, uint32_t *dense) {
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < m; i += stride) {
        uint32_t *p = dense + idx[i];
        uint32_t v;
        asm volatile("ld.global.L2::64B.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
        *p = __float_as_uint(__fadd_rn(__uint_as_float(v), 1.0f));
    }
}

cudaError_t launch_probe_rmw(const uint32_t *idx, uint64_t m, void *dense, cudaStream_t s) {
    if (m == 0) return cudaSuccess;
    uint64_t blocks = (m + 255) / 256;
    const uint64_t cap = (uint64_t)num_sms() * 8;
    if (blocks > cap) blocks = cap;
    probe_rmw_kernel<<<(unsigned)blocks, 256, 0, s>>>(idx, m, reinterpret_cast<uint32_t *>(dense));
    return cudaGetLastError();
}

}  // namespace pici
