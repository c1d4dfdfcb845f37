// host_pipeline.cu — qcd_md_host: the MD step on HOST buffers (the end-to-end number of bench.py), pipelined.
//
// The paper overlaps host<->device transfers with kernels on CUDA streams (section 5.1, Fig. 2).
// Here the lattice is cut into slabs of timeslices and three internal streams run as a pipeline:
//   up    H2D copies of slab k of U and P (canonical layout) into one of two staging buffers
//   comp  pack slab k into the device layout; the single-pass MD step on slab j as soon as its neighbours j-1, j+1
//         are packed (the stencil reaches one timeslice); unpack slab j of the result into an output staging buffer
//   down  D2H copies of the finished slabs
// so that, for a single step, both PCIe directions are busy at once and the kernels hide behind the copies.  With
// nsteps > 1 the first step overlaps the upload, the last one the download, the steps between run on the whole
// lattice.  The caller's stream is joined at entry and at exit with events; nothing synchronises the host.
#include <map>
#include <vector>

#include "qcd_internal.h"

namespace qcd {

namespace {

// The three streams and the events belong to one device, so there is one Pipe per (host thread, device): created on
// the first qcd_md_host call of that thread with that device current, reused by later calls, destroyed when the
// thread exits (for the main thread: before the CUDA runtime's own exit handlers run).
struct Pipe {
    cudaStream_t up = nullptr, comp = nullptr, down = nullptr;
    std::vector<cudaEvent_t> ev;
    size_t used = 0;
    Pipe() = default;
    Pipe(const Pipe &) = delete;
    Pipe &operator=(const Pipe &) = delete;
    ~Pipe() {
        for (cudaEvent_t e : ev) cudaEventDestroy(e);
        for (cudaStream_t s : {up, comp, down})
            if (s) cudaStreamDestroy(s);
    }
    bool ok() {
        if (up && comp && down) return true;
        return (up || cudaStreamCreateWithFlags(&up, cudaStreamNonBlocking) == cudaSuccess) &&
               (comp || cudaStreamCreateWithFlags(&comp, cudaStreamNonBlocking) == cudaSuccess) &&
               (down || cudaStreamCreateWithFlags(&down, cudaStreamNonBlocking) == cudaSuccess);
    }
    cudaEvent_t event() {  // events are reused from call to call (recording again is legal once waited on)
        if (used == ev.size()) {
            cudaEvent_t e;
            if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) return nullptr;
            ev.push_back(e);
        }
        return ev[used++];
    }
};
thread_local std::map<int, Pipe> g_pipes;  // key: device ordinal

int cuda_rc(cudaError_t e, const char *what) {
    if (e == cudaSuccess) return QCD_OK;
    set_error("qcd_md_host: %s: %s", what, cudaGetErrorString(e));
    return QCD_ECUDA;
}

#define PIPE_TRY(expr)                 \
    do {                               \
        const int rc_ = (expr);        \
        if (rc_ != QCD_OK) return rc_; \
    } while (0)

// number of slabs: the largest divisor of Lt that is <= 16; fewer than 8 slabs: no pipeline (staging would not fit)
int slab_count(int Lt) {
    int ns = 1;
    for (int d = 1; d <= 16; d++)
        if (Lt % d == 0) ns = d;
    return ns;
}

}  // namespace

bool md_host_can_pipeline(const qcd_lattice *lat) {
    return lat->p.t0 == 0 && lat->p.t1 == lat->p.L[3] && slab_count(lat->p.L[3]) >= 8;
}

// work: 4 device fields: U_a, P, U_b, staging (8 slab buffers of canonical data).  All arguments validated by the caller.
int md_host_pipelined(const qcd_lattice *lat, int prec, double beta, double eps, int nsteps, void *U_host,
                      void *P_host, void *work, size_t fb, cudaStream_t user) {
    int dev = -1;
    PIPE_TRY(cuda_rc(cudaGetDevice(&dev), "cudaGetDevice"));
    Pipe &pp = g_pipes[dev];
    if (!pp.ok()) return cuda_rc(cudaGetLastError(), "stream creation");
    pp.used = 0;
    const int Lt = lat->p.L[3], ns = slab_count(Lt), ts = Lt / ns;
    const size_t rb = prec == QCD_F64 ? 8 : 4;
    const size_t shb = (size_t)(lat->p.V / Lt) * ts * 72 * rb;  // canonical bytes of one slab of one field
    char *w = (char *)work;
    void *P = w + fb;
    void *Ubuf[2] = {w, w + 2 * fb};
    char *stage = w + 3 * fb;
    char *inU[2] = {stage, stage + 2 * shb}, *inP[2] = {stage + shb, stage + 3 * shb};
    char *outU[2] = {stage + 4 * shb, stage + 6 * shb}, *outP[2] = {stage + 5 * shb, stage + 7 * shb};

    // per-slab descriptors: the same lattice with the stencil restricted to the slab's timeslices
    std::vector<qcd_lattice> view(ns, *lat);
    for (int k = 0; k < ns; k++) {
        view[k].p.t0 = k * ts;
        view[k].p.t1 = (k + 1) * ts;
        default_force_tile(view[k].p, 2, view[k].tile_all);
    }

    cudaEvent_t e_start = pp.event();
    if (!e_start) return cuda_rc(cudaGetLastError(), "event creation");
    PIPE_TRY(cuda_rc(cudaEventRecord(e_start, user), "event record"));
    for (cudaStream_t s : {pp.up, pp.comp, pp.down}) PIPE_TRY(cuda_rc(cudaStreamWaitEvent(s, e_start, 0), "stream wait"));

    int cur = 0;  // Ubuf[cur] holds the current links
    std::vector<cudaEvent_t> e_packed(ns, nullptr);
    int nout = 0;
    cudaEvent_t e_d2h[2] = {nullptr, nullptr};

    // one slab of the LAST step: compute (unless nsteps == 0), unpack into an output buffer, copy to the host
    auto finish_slab = [&](int j, bool compute) -> int {
        if (compute)
            PIPE_TRY(launch_md_single(&view[j], prec, beta, eps, eps, Ubuf[cur], P, Ubuf[cur ^ 1], pp.comp));
        const int b = nout & 1;
        if (e_d2h[b]) PIPE_TRY(cuda_rc(cudaStreamWaitEvent(pp.comp, e_d2h[b], 0), "stream wait"));
        const void *Ures = compute ? Ubuf[cur ^ 1] : Ubuf[cur];
        PIPE_TRY(launch_pack_slab(lat, prec, 72, true, Ures, outU[b], true, j * ts, ts, pp.comp));
        PIPE_TRY(launch_pack_slab(lat, prec, 72, true, P, outP[b], true, j * ts, ts, pp.comp));
        cudaEvent_t e_unp = pp.event();
        if (!e_unp) return cuda_rc(cudaGetLastError(), "event creation");
        PIPE_TRY(cuda_rc(cudaEventRecord(e_unp, pp.comp), "event record"));
        PIPE_TRY(cuda_rc(cudaStreamWaitEvent(pp.down, e_unp, 0), "stream wait"));
        PIPE_TRY(cuda_rc(cudaMemcpyAsync((char *)U_host + (size_t)j * shb, outU[b], shb, cudaMemcpyDeviceToHost, pp.down), "D2H copy"));
        PIPE_TRY(cuda_rc(cudaMemcpyAsync((char *)P_host + (size_t)j * shb, outP[b], shb, cudaMemcpyDeviceToHost, pp.down), "D2H copy"));
        e_d2h[b] = pp.event();
        if (!e_d2h[b]) return cuda_rc(cudaGetLastError(), "event creation");
        PIPE_TRY(cuda_rc(cudaEventRecord(e_d2h[b], pp.down), "event record"));
        nout++;
        return QCD_OK;
    };
    // one slab of the FIRST step, as soon as its neighbours are on the device
    auto first_slab = [&](int j) -> int {
        if (nsteps == 1) return finish_slab(j, true);
        return launch_md_single(&view[j], prec, beta, eps, eps, Ubuf[0], P, Ubuf[1], pp.comp);
    };

    // ---- upload + first step
    for (int k = 0; k < ns; k++) {
        const int b = k & 1;
        if (k >= 2) PIPE_TRY(cuda_rc(cudaStreamWaitEvent(pp.up, e_packed[k - 2], 0), "stream wait"));
        PIPE_TRY(cuda_rc(cudaMemcpyAsync(inU[b], (const char *)U_host + (size_t)k * shb, shb, cudaMemcpyHostToDevice, pp.up), "H2D copy"));
        PIPE_TRY(cuda_rc(cudaMemcpyAsync(inP[b], (const char *)P_host + (size_t)k * shb, shb, cudaMemcpyHostToDevice, pp.up), "H2D copy"));
        cudaEvent_t e_h2d = pp.event();
        if (!e_h2d) return cuda_rc(cudaGetLastError(), "event creation");
        PIPE_TRY(cuda_rc(cudaEventRecord(e_h2d, pp.up), "event record"));
        PIPE_TRY(cuda_rc(cudaStreamWaitEvent(pp.comp, e_h2d, 0), "stream wait"));
        PIPE_TRY(launch_pack_slab(lat, prec, 72, true, inU[b], Ubuf[0], false, k * ts, ts, pp.comp));
        PIPE_TRY(launch_pack_slab(lat, prec, 72, true, inP[b], P, false, k * ts, ts, pp.comp));
        e_packed[k] = pp.event();
        if (!e_packed[k]) return cuda_rc(cudaGetLastError(), "event creation");
        PIPE_TRY(cuda_rc(cudaEventRecord(e_packed[k], pp.comp), "event record"));
        if (nsteps >= 1 && k >= 2) PIPE_TRY(first_slab(k - 1));  // slabs k-2, k-1, k are packed (same stream: in order)
    }
    if (nsteps >= 1) {
        PIPE_TRY(first_slab(ns - 1));  // periodic wrap: the first and the last slab need each other
        PIPE_TRY(first_slab(0));
        if (nsteps > 1) cur = 1;
    }
    // ---- steps between the first and the last, whole lattice
    for (int s = 1; s + 1 < nsteps; s++) {
        PIPE_TRY(launch_md_single(lat, prec, beta, eps, eps, Ubuf[cur], P, Ubuf[cur ^ 1], pp.comp));
        cur ^= 1;
    }
    // ---- last step + download (nsteps == 1: done above; nsteps == 0: round trip only)
    if (nsteps != 1)
        for (int j = 0; j < ns; j++) PIPE_TRY(finish_slab(j, nsteps > 1));

    // ---- join the caller's stream
    cudaEvent_t e_comp = pp.event(), e_down = pp.event();
    if (!e_comp || !e_down) return cuda_rc(cudaGetLastError(), "event creation");
    PIPE_TRY(cuda_rc(cudaEventRecord(e_comp, pp.comp), "event record"));
    PIPE_TRY(cuda_rc(cudaEventRecord(e_down, pp.down), "event record"));
    PIPE_TRY(cuda_rc(cudaStreamWaitEvent(user, e_comp, 0), "stream wait"));
    return cuda_rc(cudaStreamWaitEvent(user, e_down, 0), "stream wait");
}

}  // namespace qcd
