// ring.cu - SpCCL's sparse ring collectives over P LOGICAL ranks held in one B200's HBM, enqueued from C
// (include/pici.h "Ring engine"; PAPER.md:207-219 ring AG / RS / AR, 227-247 the
// dense switch and the adaptive policy).  No NCCL and no inter-GPU traffic (north_star): a "send" is a pointer
// hand-off between slots of the caller's arena.
//
// One ring step of ALL ranks is one launch per kernel family (launch.h: a batch of P jobs, block (x, y) works
// on rank y's job), so a step costs a handful of launches whatever P is, and nothing is read back: every
// format decision is taken ON THE DEVICE and steers the next kernels through gate words.
//   decision = MEASURED: a message travels dense once its measured nnz reaches nnz_switch (pici_maybe_densify;
//              the reading of C9 #9/#10); once dense it stays dense within the reduce-scatter.
//   decision = POLICY:   the paper's rule: every rank tracks one sparsity; a send is dense
//              when sigma_prev * sigma_0 (Eq. 7) is <= the threshold of the link it goes over (intra / inter
//              node), a dense send carries the extrapolation forward, a compression re-calibrates it with the
//              computed count; ag_thresh decides the all-gather phase of an all-reduce.  ring_policy_kernel
//              holds that state machine (fp64, the oracle's expressions) and writes a CODE word per (step, rank):
//              code = format of the incoming message + 2 * format of the outgoing one.
// Schedule (NCCL's; C8): rank r sends to r + 1 and ends owning chunk r; reduce-scatter step 0 encodes chunk
// (r - 1) mod P; at step s rank r receives chunk (r - 1 - s) mod P and forms acc = received + local.
#include <new>

#include "launch.h"
#include "pici_common.cuh"
#include "../../include/pici.h"

namespace pici {

namespace {

constexpr uint32_t kNoCount = 0xFFFFFFFFu;   // nnz log of a dense send: no count was computed

inline uint64_t up(uint64_t v, uint64_t a) { return (v + a - 1) / a * a; }

// Where everything lives inside the caller's arena (byte offsets; every region 256-byte aligned).
struct Layout {
    int P;
    uint64_t n, T;
    uint64_t ws_bytes, b_bytes, i_bytes, a_bytes, pici_bytes, msg_bytes;
    uint64_t off_log_fmt, off_log_nnz, off_log_sigma, off_code, off_state;   // logs and policy state
    uint64_t off_ws, off_local, off_reduced, off_msgs;
    uint64_t rs_records, records, slots, total;
    bool keep;

    Layout(const pici_ring_config &c) {
        P = c.ranks;
        n = c.chunk;
        T = n / kTile;
        keep = c.keep_messages != 0;
        ws_bytes = up(scan_workspace_bytes(n), 256);
        b_bytes = up(64 * T * 8, 256);
        i_bytes = up((T + 1) * 4, 256);
        a_bytes = up(n * 4, 256);
        pici_bytes = b_bytes + i_bytes + a_bytes;
        msg_bytes = pici_bytes + a_bytes;                       // a message slot: Pici form + dense form
        rs_records = (uint64_t)(P - 1) * P;                     // reduce-scatter: steps 0 .. P-2, every rank
        records = rs_records + P;                               // + the all-gather's step-0 messages
        slots = keep ? records : 3ull * P;                      // else: two alternating sets for RS, one for AG
        uint64_t o = 0;
        off_log_fmt = o;   o += up(records * 4, 256);
        off_log_nnz = o;   o += up(records * 4, 256);
        off_log_sigma = o; o += up(records * 8, 256);
        off_code = o;      o += up(((uint64_t)P * P) * 4, 256);
        off_state = o;     o += up((uint64_t)P * 16, 256);
        off_ws = o;        o += (uint64_t)P * ws_bytes;
        off_local = o;     o += (uint64_t)P * pici_bytes;
        off_reduced = o;   o += (uint64_t)P * a_bytes;
        off_msgs = o;      o += slots * msg_bytes;
        total = o;
    }
    uint64_t rs_rec(int step, int r) const { return (uint64_t)step * P + r; }
    uint64_t ag_rec(int r) const { return rs_records + r; }
    uint64_t rs_slot(int step, int r) const { return keep ? rs_rec(step, r) : (uint64_t)(step & 1) * P + r; }
    uint64_t ag_slot(int r) const { return keep ? ag_rec(r) : 2ull * P + r; }
};

struct PiciPtrs {
    uint64_t *B;
    uint32_t *I;
    uint32_t *A;
};

struct Arena {
    const Layout &L;
    unsigned char *base;
    Arena(const Layout &l, void *p) : L(l), base(static_cast<unsigned char *>(p)) {}
    int32_t *fmt(uint64_t rec) const { return reinterpret_cast<int32_t *>(base + L.off_log_fmt) + rec; }
    uint32_t *nnz(uint64_t rec) const { return reinterpret_cast<uint32_t *>(base + L.off_log_nnz) + rec; }
    double *sigma_log(uint64_t rec) const { return reinterpret_cast<double *>(base + L.off_log_sigma) + rec; }
    int32_t *code(int step, int r) const { return reinterpret_cast<int32_t *>(base + L.off_code) + (uint64_t)step * L.P + r; }
    double *state() const { return reinterpret_cast<double *>(base + L.off_state); }   // [P] sigma_0, [P] sigma
    void *ws(int r) const { return base + L.off_ws + (uint64_t)r * L.ws_bytes; }
    PiciPtrs pici_at(uint64_t off) const {
        return {reinterpret_cast<uint64_t *>(base + off), reinterpret_cast<uint32_t *>(base + off + L.b_bytes),
                reinterpret_cast<uint32_t *>(base + off + L.b_bytes + L.i_bytes)};
    }
    PiciPtrs local(int r) const { return pici_at(L.off_local + (uint64_t)r * L.pici_bytes); }
    float *reduced(int r) const { return reinterpret_cast<float *>(base + L.off_reduced + (uint64_t)r * L.a_bytes); }
    PiciPtrs msg_pici(uint64_t slot) const { return pici_at(L.off_msgs + slot * L.msg_bytes); }
    float *msg_dense(uint64_t slot) const { return reinterpret_cast<float *>(base + L.off_msgs + slot * L.msg_bytes + L.pici_bytes); }
};

// ---- the paper's policy on the device (oracle/ring_oracle.py ring_reduce_scatter_policy) ----
struct PolicyRank {
    const uint32_t *I_prev;   // index array of this rank's previous message (its I[T] calibrates), or nullptr
    const int32_t *fmt_prev;  // format word of this rank's previous message
    uint32_t *nnz_prev;       // nnz log entry of that message
    const int32_t *fmt_in;    // format word of the message received at this step (nullptr at step 0)
    int32_t *fmt_out;         // format word of the message sent at this step (nullptr at the last step)
    double *sigma_log;        // the sparsity the decision is taken on
    int32_t *code;            // fmt_in + 2 * fmt_out (nullptr at step 0)
    double thresh;            // threshold of the rank's outgoing link
};
struct PolicyStep {
    PolicyRank rank[kMaxBatch];
    double *state;            // [P] sigma_0 then [P] sigma
    uint64_t n;
    uint32_t T;
    int P, kind;              // kind 0: step 0; 1: intermediate; 2: last reduce-scatter step; 3: RS -> AG transition
};
__global__ void ring_policy_kernel(const PolicyStep s) {
    const int r = threadIdx.x;
    if (r >= s.P) return;
    const PolicyRank &q = s.rank[r];
    double *sigma0 = s.state + r, *sigma = s.state + s.P + r;
    const double nd = (double)s.n;
    if (s.kind == 0) {   // step 0 always compresses; the decision is taken on the computed sparsity
        const uint32_t nnz = q.I_prev[s.T];
        const double sg = __dsub_rn(1.0, __ddiv_rn((double)nnz, nd));
        *sigma0 = *sigma = sg;
        const int out = sg <= q.thresh ? PICI_FMT_DENSE : PICI_FMT_PICI;
        *q.fmt_out = out;
        *q.sigma_log = sg;
        *q.nnz_prev = out == PICI_FMT_PICI ? nnz : kNoCount;
        return;
    }
    if (s.kind == 3) {   // ag_thresh on the tracked sparsity
        const double sg = *sigma;
        *q.fmt_out = sg <= q.thresh ? PICI_FMT_DENSE : PICI_FMT_PICI;
        *q.sigma_log = sg;
        return;
    }
    // a compression at the previous step calibrates the tracked sparsity with its count
    double sg = *sigma;
    if (q.I_prev != nullptr) {
        if (*q.fmt_prev == PICI_FMT_PICI) {
            const uint32_t nnz = q.I_prev[s.T];
            sg = __dsub_rn(1.0, __ddiv_rn((double)nnz, nd));
            *q.nnz_prev = nnz;
        } else {
            *q.nnz_prev = kNoCount;
        }
    }
    const double ext = __dmul_rn(sg, *sigma0);   // Eq. 7
    if (s.kind == 2) {                           // last step: the accumulation is the rank's output
        *sigma = ext;
        return;
    }
    const int out = ext <= q.thresh ? PICI_FMT_DENSE : PICI_FMT_PICI;
    *sigma = out == PICI_FMT_DENSE ? ext : sg;   // a dense send carries the extrapolation; a sparse one is calibrated next step
    *q.fmt_out = out;
    *q.sigma_log = ext;
    *q.code = *q.fmt_in + 2 * out;
}

// nnz log of the measured mode: I[T] of a Pici message, kNoCount where the chunk travels dense.
struct LogStep {
    const uint32_t *I[kMaxBatch];
    const int32_t *fmt_in[kMaxBatch];   // nullptr: always count
    uint32_t *nnz[kMaxBatch];
    uint32_t T;
    int P;
};
__global__ void ring_log_kernel(const LogStep s) {
    const int r = threadIdx.x;
    if (r >= s.P) return;
    const bool sparse = s.fmt_in[r] == nullptr || *s.fmt_in[r] == PICI_FMT_PICI;
    *s.nnz[r] = sparse ? s.I[r][s.T] : kNoCount;
}

struct Engine {
    const pici_ring_config &c;
    Layout L;
    Arena a;
    cudaStream_t st;
    cudaError_t err = cudaSuccess;
    int launches = 0;
    bool policy, paper;

    Engine(const pici_ring_config &cfg, void *arena, cudaStream_t s)
        : c(cfg), L(cfg), a(L, arena), st(s), policy(cfg.decision == PICI_RING_DECIDE_POLICY),
          paper(cfg.strategy == PICI_RING_PAPER) {}

    void ok(cudaError_t e) {
        ++launches;
        if (err == cudaSuccess) err = e;
    }
    double link_thresh(int r) const {
        const int rpn = c.ranks_per_node > 0 ? c.ranks_per_node : 1;
        const bool same = (r / rpn) == (((r + 1) % L.P) / rpn);
        return same ? c.intra_thresh : c.inter_thresh;
    }
    const float *chunk(const void *const *X, int r, int ch) const { return static_cast<const float *>(X[r]) + (uint64_t)ch * L.n; }

    // ---- reduce-scatter: out[r] = reduced chunk r (n elements) -------------------------------------------------
    void reduce_scatter(const void *const *X, void *const *out) {
        const int P = L.P;
        const uint64_t n = L.n;
        CompressJob cj[kMaxBatch];
        ExpandJob ej[kMaxBatch];
        MergeJob mj[kMaxBatch];
        DenseAddJob aj[kMaxBatch];
        DenseCopyJob dj[kMaxBatch];
        const Gate open = {nullptr, 0, 0};
        // ---- step 0: every rank compresses chunk (r - 1) mod P of its own input ----
        for (int r = 0; r < P; ++r) {
            const PiciPtrs m = a.msg_pici(L.rs_slot(0, r));
            cj[r] = {chunk(X, r, (r + P - 1) % P), n, m.B, m.I, m.A, a.ws(r), open};
        }
        ok(launch_compress_batch(cj, P, PICI_F32, st));
        if (policy) {
            PolicyStep ps = {};
            for (int r = 0; r < P; ++r) {
                const uint64_t rec = L.rs_rec(0, r);
                ps.rank[r] = {a.msg_pici(L.rs_slot(0, r)).I, nullptr, a.nnz(rec), nullptr, a.fmt(rec), a.sigma_log(rec), nullptr,
                              link_thresh(r)};
                dj[r] = {chunk(X, r, (r + P - 1) % P), a.msg_dense(L.rs_slot(0, r)), n * 4, gate_eq(a.fmt(rec), PICI_FMT_DENSE)};
            }
            ps.state = a.state(); ps.n = n; ps.T = (uint32_t)L.T; ps.P = P; ps.kind = 0;
            ring_policy_kernel<<<1, 32, 0, st>>>(ps);
            ok(cudaGetLastError());
            ok(launch_dense_copy_batch(dj, P, st));
        } else {
            LogStep ls = {};
            for (int r = 0; r < P; ++r) {
                const uint64_t rec = L.rs_rec(0, r), slot = L.rs_slot(0, r);
                const PiciPtrs m = a.msg_pici(slot);
                ej[r] = {m.B, m.I, m.A, n, nullptr, a.msg_dense(slot), DensifyCtl{a.fmt(rec), c.nnz_switch_rs, PICI_FMT_DENSE, PICI_FMT_PICI}, open};
                ls.I[r] = m.I; ls.fmt_in[r] = nullptr; ls.nnz[r] = a.nnz(rec);
            }
            ok(launch_expand_batch(ej, P, PICI_F32, 0, st));
            ls.T = (uint32_t)L.T; ls.P = P;
            ring_log_kernel<<<1, 32, 0, st>>>(ls);
            ok(cudaGetLastError());
        }
        // ---- steps 1 .. P-1 ----
        for (int s = 1; s < P; ++s) {
            const bool last = s == P - 1;
            if (policy) {
                PolicyStep ps = {};
                for (int r = 0; r < P; ++r) {
                    const int from = (r + P - 1) % P;
                    const uint64_t prev = L.rs_rec(s - 1, r), rec = L.rs_rec(s, r);
                    PolicyRank &q = ps.rank[r];
                    q.I_prev = s - 1 >= 1 ? a.msg_pici(L.rs_slot(s - 1, r)).I : nullptr;   // step 0's count is sigma_0 itself
                    q.fmt_prev = a.fmt(prev);
                    q.nnz_prev = a.nnz(prev);
                    q.fmt_in = a.fmt(L.rs_rec(s - 1, from));
                    q.fmt_out = last ? nullptr : a.fmt(rec);
                    q.sigma_log = last ? nullptr : a.sigma_log(rec);
                    q.code = last ? nullptr : a.code(s, r);
                    q.thresh = link_thresh(r);
                }
                ps.state = a.state(); ps.n = n; ps.T = (uint32_t)L.T; ps.P = P; ps.kind = last ? 2 : 1;
                ring_policy_kernel<<<1, 32, 0, st>>>(ps);
                ok(cudaGetLastError());
            }
            if (last) {   // acc = received + local is rank r's dense output
                for (int r = 0; r < P; ++r) {
                    const int from = (r + P - 1) % P, ch = (r + 2 * P - 1 - s) % P;
                    const uint64_t slot = L.rs_slot(s - 1, from);
                    const int32_t *f_in = a.fmt(L.rs_rec(s - 1, from));
                    const PiciPtrs mi = a.msg_pici(slot);
                    ej[r] = {mi.B, mi.I, mi.A, n, chunk(X, r, ch), out[r], DensifyCtl{nullptr, 0, 0, 0}, gate_eq(f_in, PICI_FMT_PICI)};
                    aj[r] = {a.msg_dense(slot), chunk(X, r, ch), n, out[r], nullptr, gate_eq(f_in, PICI_FMT_DENSE)};
                }
                ok(launch_expand_batch(ej, P, PICI_F32, 1, st));
                ok(launch_dense_add_batch(aj, P, st));
                break;
            }
            CompressJob cj2[kMaxBatch];
            LogStep ls = {};
            for (int r = 0; r < P; ++r) {
                const int from = (r + P - 1) % P, ch = (r + 2 * P - 1 - s) % P;
                const uint64_t slot_in = L.rs_slot(s - 1, from), slot = L.rs_slot(s, r), rec = L.rs_rec(s, r);
                const int32_t *f_in = a.fmt(L.rs_rec(s - 1, from));
                const PiciPtrs mi = a.msg_pici(slot_in), mo = a.msg_pici(slot), lo = a.local(r);
                const float *loc = chunk(X, r, ch);
                float *md = a.msg_dense(slot);
                const int32_t *cw = a.code(s, r);
                // gates.  measured: the incoming format; policy: the code word (incoming + 2 * outgoing)
                Gate g_pp = gate_eq(f_in, PICI_FMT_PICI);         // sparse in, sparse out
                Gate g_sparse_in = g_pp, g_dense_in = gate_eq(f_in, PICI_FMT_DENSE);
                Gate g_pd = {f_in, 0, 1}, g_dp = {f_in, 0, 1};    // never open in measured mode
                Gate g_out_sparse = g_pp;
                if (policy) {
                    g_pp = gate_eq(cw, 0);
                    g_sparse_in = Gate{cw, 1, 0};
                    g_dense_in = Gate{cw, 1, 1};
                    g_pd = gate_eq(cw, 2);                        // sparse in, dense out
                    g_dp = gate_eq(cw, 1);                        // dense in, sparse out (the sandwich)
                    g_out_sparse = Gate{cw, 2, 0};
                }
                const DensifyCtl no_ctl = {nullptr, 0, 0, 0};
                if (!paper) {
                    const CompressJob c1 = {loc, n, lo.B, lo.I, lo.A, a.ws(r), g_pp};
                    const MergeJob m1 = {mi.B, mi.I, mi.A, lo.B, lo.I, lo.A, n, mo.B, mo.I, mo.A, a.ws(r), g_pp};
                    const ExpandJob e1 = {mi.B, mi.I, mi.A, n, loc, md, no_ctl, g_pd};   // scatter-add into the dense form
                    const CompressJob c2 = {md, n, mo.B, mo.I, mo.A, a.ws(r), g_dp};     // dense add, then compress the sum
                    cj[r] = c1; mj[r] = m1; ej[r] = e1; cj2[r] = c2;
                } else {
                    const ExpandJob e1 = {mi.B, mi.I, mi.A, n, loc, md, no_ctl, g_sparse_in};
                    const CompressJob c2 = {md, n, mo.B, mo.I, mo.A, a.ws(r), g_out_sparse};   // recompress the accumulation
                    ej[r] = e1; cj2[r] = c2;
                }
                int32_t *fmt_out = policy ? nullptr : a.fmt(rec);
                const DenseAddJob a1 = {a.msg_dense(slot_in), loc, n, md, fmt_out, g_dense_in};
                aj[r] = a1;
                ls.I[r] = mo.I; ls.fmt_in[r] = f_in; ls.nnz[r] = a.nnz(rec);
            }
            if (!paper) {
                ok(launch_compress_batch(cj, P, PICI_F32, st));
                ok(launch_reduce_ss_batch(mj, P, st));
                if (policy) ok(launch_expand_batch(ej, P, PICI_F32, 1, st));
            } else {
                ok(launch_expand_batch(ej, P, PICI_F32, 1, st));
            }
            ok(launch_dense_add_batch(aj, P, st));
            if (paper || policy) ok(launch_compress_batch(cj2, P, PICI_F32, st));
            if (!policy) {   // measured: decide on the count of the new message, log it
                for (int r = 0; r < P; ++r) {
                    const int from = (r + P - 1) % P;
                    const uint64_t slot = L.rs_slot(s, r), rec = L.rs_rec(s, r);
                    const PiciPtrs mo = a.msg_pici(slot);
                    ej[r] = {mo.B, mo.I, mo.A, n, nullptr, paper ? nullptr : a.msg_dense(slot),
                             DensifyCtl{a.fmt(rec), c.nnz_switch_rs, PICI_FMT_DENSE, PICI_FMT_PICI},
                             gate_eq(a.fmt(L.rs_rec(s - 1, from)), PICI_FMT_PICI)};
                }
                ok(launch_expand_batch(ej, P, PICI_F32, 0, st));
                ls.T = (uint32_t)L.T; ls.P = P;
                ring_log_kernel<<<1, 32, 0, st>>>(ls);
                ok(cudaGetLastError());
            }
        }
    }

    // ---- all-gather: out[r] = the P shards in order (P * n elements) ------------------------------------------------
    // from_reduce: the shards are the reduced chunks of an all-reduce and, in policy mode, ag_thresh decides (kind 3)
    void all_gather(const void *const *shards, void *const *out, bool from_reduce) {
        const int P = L.P;
        const uint64_t n = L.n;
        CompressJob cj[kMaxBatch];
        ExpandJob ej[kMaxBatch];
        DenseCopyJob dj[kMaxBatch];
        const Gate open = {nullptr, 0, 0};
        const bool pol = policy && from_reduce;
        if (pol) {
            PolicyStep ps = {};
            for (int r = 0; r < P; ++r) {
                ps.rank[r] = {};
                ps.rank[r].fmt_out = a.fmt(L.ag_rec(r));
                ps.rank[r].sigma_log = a.sigma_log(L.ag_rec(r));
                ps.rank[r].thresh = c.ag_thresh;
            }
            ps.state = a.state(); ps.n = n; ps.T = (uint32_t)L.T; ps.P = P; ps.kind = 3;
            ring_policy_kernel<<<1, 32, 0, st>>>(ps);
            ok(cudaGetLastError());
        }
        LogStep ls = {};
        for (int r = 0; r < P; ++r) {   // step 0: compress once; own slot: plain copy (C9 #12)
            const uint64_t slot = L.ag_slot(r), rec = L.ag_rec(r);
            const PiciPtrs m = a.msg_pici(slot);
            cj[r] = {shards[r], n, m.B, m.I, m.A, a.ws(r), pol ? gate_eq(a.fmt(rec), PICI_FMT_PICI) : open};
            ej[r] = {m.B, m.I, m.A, n, nullptr, nullptr, DensifyCtl{a.fmt(rec), c.nnz_switch_ag, PICI_FMT_DENSE, PICI_FMT_PICI}, open};
            dj[r] = {shards[r], static_cast<float *>(out[r]) + (uint64_t)r * n, n * 4, open};
            ls.I[r] = m.I; ls.fmt_in[r] = pol ? a.fmt(rec) : nullptr; ls.nnz[r] = a.nnz(rec);
        }
        ok(launch_compress_batch(cj, P, PICI_F32, st));
        if (!pol) ok(launch_expand_batch(ej, P, PICI_F32, 0, st));   // flag only: a dense message aliases the shard
        ls.T = (uint32_t)L.T; ls.P = P;
        ring_log_kernel<<<1, 32, 0, st>>>(ls);
        ok(cudaGetLastError());
        ok(launch_dense_copy_batch(dj, P, st));
        for (int s = 1; s < P; ++s) {   // forwarded unchanged; every received shard is decompressed at once
            for (int r = 0; r < P; ++r) {
                const int ch = (r + P - s) % P;
                const PiciPtrs m = a.msg_pici(L.ag_slot(ch));
                float *slot = static_cast<float *>(out[r]) + (uint64_t)ch * n;
                const int32_t *f = a.fmt(L.ag_rec(ch));
                ej[r] = {m.B, m.I, m.A, n, nullptr, slot, DensifyCtl{nullptr, 0, 0, 0}, gate_eq(f, PICI_FMT_PICI)};
                dj[r] = {shards[ch], slot, n * 4, gate_eq(f, PICI_FMT_DENSE)};
            }
            ok(launch_expand_batch(ej, P, PICI_F32, 0, st));
            ok(launch_dense_copy_batch(dj, P, st));
        }
    }
};

int check(const pici_ring_config *c, const void *arena, uint64_t arena_bytes) {
    if (c == nullptr) return PICI_ERR_INVALID_ARG;
    if (c->ranks < 2 || c->ranks > kMaxBatch || c->chunk == 0 || c->chunk % kTile != 0 || c->chunk >= (1ull << 32))
        return PICI_ERR_INVALID_ARG;
    if ((c->strategy != PICI_RING_FUSED && c->strategy != PICI_RING_PAPER) ||
        (c->decision != PICI_RING_DECIDE_MEASURED && c->decision != PICI_RING_DECIDE_POLICY))
        return PICI_ERR_INVALID_ARG;
    if (arena == nullptr) return PICI_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(arena) & 255u) != 0) return PICI_ERR_ALIGN;
    if (arena_bytes < Layout(*c).total) return PICI_ERR_WORKSPACE;
    return PICI_OK;
}

int check_ptrs(const void *const *p, int count) {
    if (p == nullptr) return PICI_ERR_INVALID_ARG;
    for (int i = 0; i < count; ++i) {
        if (p[i] == nullptr) return PICI_ERR_INVALID_ARG;
        if ((reinterpret_cast<uintptr_t>(p[i]) & 15u) != 0) return PICI_ERR_ALIGN;
    }
    return PICI_OK;
}

}  // namespace
}  // namespace pici

using namespace pici;

extern "C" {

int pici_ring_arena_bytes(const pici_ring_config *cfg, uint64_t *bytes) {
    if (cfg == nullptr || bytes == nullptr || cfg->ranks < 2 || cfg->ranks > kMaxBatch || cfg->chunk == 0 ||
        cfg->chunk % kTile != 0 || cfg->chunk >= (1ull << 32))
        return PICI_ERR_INVALID_ARG;
    *bytes = Layout(*cfg).total;
    return PICI_OK;
}

int pici_ring_layout(const pici_ring_config *cfg, pici_ring_layout_info *info) {
    if (cfg == nullptr || info == nullptr || cfg->ranks < 2 || cfg->ranks > kMaxBatch || cfg->chunk == 0 ||
        cfg->chunk % kTile != 0 || cfg->chunk >= (1ull << 32))
        return PICI_ERR_INVALID_ARG;
    const Layout L(*cfg);
    info->records = L.records;
    info->rs_records = L.rs_records;
    info->off_fmt = L.off_log_fmt;
    info->off_nnz = L.off_log_nnz;
    info->off_sigma = L.off_log_sigma;
    info->off_messages = L.off_msgs;
    info->message_bytes = L.msg_bytes;
    info->message_I = L.b_bytes;
    info->message_A = L.b_bytes + L.i_bytes;
    info->message_dense = L.pici_bytes;
    info->off_reduced = L.off_reduced;
    info->reduced_bytes = L.a_bytes;
    info->slots = L.slots;
    return PICI_OK;
}

static int finish(const Engine &e, int *h_launches) {
    if (h_launches != nullptr) *h_launches = e.launches;
    return e.err == cudaSuccess ? PICI_OK : PICI_ERR_CUDA;
}

int pici_ring_reduce_scatter(const pici_ring_config *cfg, const void *const *X, void *const *out, void *arena,
                             uint64_t arena_bytes, int *h_launches, void *stream) {
    int rc = check(cfg, arena, arena_bytes);
    if (rc == PICI_OK) rc = check_ptrs(X, cfg->ranks);
    if (rc == PICI_OK) rc = check_ptrs(out, cfg->ranks);
    if (rc != PICI_OK) return rc;
    Engine e(*cfg, arena, static_cast<cudaStream_t>(stream));
    e.reduce_scatter(X, out);
    return finish(e, h_launches);
}

int pici_ring_all_gather(const pici_ring_config *cfg, const void *const *shards, void *const *out, void *arena,
                         uint64_t arena_bytes, int *h_launches, void *stream) {
    int rc = check(cfg, arena, arena_bytes);
    if (rc == PICI_OK) rc = check_ptrs(shards, cfg->ranks);
    if (rc == PICI_OK) rc = check_ptrs(out, cfg->ranks);
    if (rc != PICI_OK) return rc;
    Engine e(*cfg, arena, static_cast<cudaStream_t>(stream));
    e.all_gather(shards, out, false);
    return finish(e, h_launches);
}

int pici_ring_all_reduce(const pici_ring_config *cfg, const void *const *X, void *const *out, void *arena,
                         uint64_t arena_bytes, int *h_launches, void *stream) {
    int rc = check(cfg, arena, arena_bytes);
    if (rc == PICI_OK) rc = check_ptrs(X, cfg->ranks);
    if (rc == PICI_OK) rc = check_ptrs(out, cfg->ranks);
    if (rc != PICI_OK) return rc;
    Engine e(*cfg, arena, static_cast<cudaStream_t>(stream));
    void *red[kMaxBatch];
    for (int r = 0; r < cfg->ranks; ++r) red[r] = e.a.reduced(r);
    e.reduce_scatter(X, red);
    e.all_gather(red, out, true);
    return finish(e, h_launches);
}

}  // extern "C"
