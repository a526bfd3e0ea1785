// mcb200.cu -- host side of libmcb200.so: the C ABI declared in include/mcb200.h.
// Build: paper_1602_05716_b200/build.py (nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -fmad=false; this file plus
// sweep_inst.cu once per pair-distance form, linked into one shared object)
#include "../../include/mcb200.h"

#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "aux_kernels.cuh"
#include "sweep_launch.h"

using namespace mcb;

namespace {

thread_local std::string g_err;

int fail(int code, const std::string& msg) {
    g_err = msg;
    return code;
}

#define CUDA_TRY(expr)                                                                           \
    do {                                                                                         \
        cudaError_t e_ = (expr);                                                                 \
        if (e_ != cudaSuccess)                                                                   \
            return fail(MC_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(e_));           \
    } while (0)

constexpr size_t kAlign = 256;
constexpr size_t kDbgWords = 16 + 1024;   // diagnostic counters of the sweep kernel (mc_debug_counters)
size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

struct Layout {
    size_t xy, zq, hh, lbq, txy, tz, lnu, wall, Dblk, OVold, OVnew, log_dE, log_flags,
        st, epart, centres, ccount, stage_pos, S1, S2, ovc, nn, sy, gbar, uc, dbg, hcode, hcount, hcursor, hsxy, hszq, hbbox, total;
};

int padded(int64_t N) { return (int)((N + kTile - 1) / kTile * kTile); }

Layout make_layout(int64_t N) {
    Layout L{};
    const size_t Np = (size_t)padded(N);
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
    const size_t nt = kChunkMax / kTile;
    L.xy = take(Np * 16); L.zq = take(Np * 16); L.hh = take(Np * 8); L.lbq = take(Np * 8);
    L.txy = take(Np * 16); L.tz = take(Np * 8); L.lnu = take(Np * 8); L.wall = take(Np);
    // a ring of kDRing buffers by chunk index (the sweep kernel prepares the next chunks while the chain is in c)
    L.Dblk = take((size_t)kDRing * (nt * (nt + 1) / 2) * kTile * kTile * 8);
    L.OVold = take((size_t)kDRing * kChunkMax * nt * 4); L.OVnew = take((size_t)kDRing * kChunkMax * nt * 4);
    L.S1 = take(Np * 8); L.S2 = take(Np * 8); L.ovc = take(Np * 4); L.nn = take(Np * 8);
    L.sy = take((size_t)2 * (kSyHdr + 4 * (Np / 256 + 1)) * 4);   // live words + snapshot of the last completed sweep
    L.gbar = take(256);
    L.uc = take(((size_t)(Np / 256 + 2) * (kChunkMax / kGroup + 1) + 16) * 4);   // urgent_units() at the smallest chunk size, rounded up
    L.dbg = take(kDbgWords * 8);
    L.hcode = take(Np * 4); L.hcount = take((size_t)kCells * 4); L.hcursor = take((size_t)kCells * 4);
    L.hsxy = take(Np * 16); L.hszq = take(Np * 16); L.hbbox = take((Np / 256 + 1) * 4 * 6 * 8);
    L.log_dE = take(Np * 8); L.log_flags = take(Np);
    L.st = take(sizeof(DevState));
    L.epart = take(((size_t)energy_units((int)Np) + 2) * 8);
    L.centres = take(Np * 4); L.ccount = take(16);
    L.stage_pos = take(3 * (size_t)N * 8);
    L.total = off;
    return L;
}

}  // namespace


struct mc_handle {
    Params p{};
    Layout L{};
    char* ws = nullptr;
    cudaStream_t stream = nullptr;
    int num_sms = 148;
    int prows = 4;           // rows per consumer thread of the sweep kernel (chunk = 256 * prows)
    int pfarcols = 256;      // columns per FAR item of the sweep kernel
    int fixcols = 0;         // columns per FIX item of the sweep kernel (0: by N)
    int dsplit = 0;          // warps per DIAG unit of the sweep kernel (0: by N)
    int erows = 4;           // rows per thread of k_energy (Gram form)
    int hist_slices = 64;   // column slices (grid.y) of k_hist
    int pmode = 0;           // 1: throughput probe (diagnostic, needs "debug"; the sweep's results are meaningless)
    bool pwave = true;       // round the FAR items of a chunk to a multiple of the FAR workers
    int pnear = 4;           // worker CTAs of the sweep kernel that serve urgent and DIAG items only
    bool debug = false;      // collect the cycle counters of mc_debug_counters
    int max_ctas = 0;        // upper limit on the CTAs of the sweep kernel (0: two per SM); small systems synchronise faster on a smaller grid
    int pgrid = 0;           // CTAs of the sweep kernel
    int pgrid_key = -1;      // (form, rows, uniform) the grid was sized and the kernel configured for
    bool uniform_d = false;  // all diameters equal: s_ij^2 is one constant
    bool allow_uniform = true;
    bool all_d_equal = false;
    int form_auto = kFormGram;   // pair-distance form the geometry allows (mc_init)
    int form = kFormGram;        // form in use (option "form": the automatic one or a more exact one)
    uint64_t launches = 0;
    double* epart = nullptr;
    int* centres = nullptr;
    int* ccount = nullptr;
    double* stage_pos = nullptr;
};

namespace {

// geometry limits of the pair-distance forms (persist.cuh)
constexpr double kGramMaxRatio = 128.0;   // GRAM  needs cavity_R / d_min <= 128 (measured: 2e-12 there, 6e-11 at 500)
constexpr double kDiffWMaxRatio = 64.0;   // DIFFW needs max_disp / d_min <= 64

// One cooperative launch that runs nsweeps full sweeps (a1-a4 each): trial generation, the pair sums, the
// sequential resolution and the commit all happen inside k_sweep (persist.cuh).
int launch_sweep(mc_handle* h, cudaStream_t s, int nsweeps) {
    SweepLaunch L{};
    L.rows = h->prows;
    L.uniform = h->uniform_d;
    L.stream = s;
    auto fn = h->form == kFormGram ? launch_sweep_gram : h->form == kFormDiffW ? launch_sweep_diffw : launch_sweep_canon;
    const int key = h->form * 16 + h->prows * 2 + (h->uniform_d ? 1 : 0);
    if (h->pgrid_key != key) {
        int occ = 0;
        L.grid = 0;
        const cudaError_t e = (cudaError_t)fn(L, &occ);
        if (e != cudaSuccess) return fail(MC_ECUDA, std::string("k_sweep configuration: ") + cudaGetErrorString(e));
        if (occ < 1) return fail(MC_ECUDA, "k_sweep does not fit on an SM");
        h->pgrid = std::min(occ, 2) * h->num_sms;
        if (h->max_ctas > 0) h->pgrid = std::max(8, std::min(h->pgrid, h->max_ctas));
        h->pgrid_key = key;
    }
    PArgs& a = L.args;
    a.p = h->p;
    a.C = 256 * h->prows;
    a.p.chunk = a.C;
    a.nchunks = (a.p.Np + a.C - 1) / a.C;
    a.nnear = std::min(h->pnear, std::max(0, h->pgrid - 4));
    a.farcols = h->pfarcols;
    a.mode = h->pmode;
    a.nfar = h->pwave ? std::max(1, h->pgrid - 2 - a.nnear) : 0;
    a.dsplit = h->dsplit > 0 ? h->dsplit : (a.p.Np <= 768 ? 4 : a.p.Np <= 6144 ? 2 : 1);
    a.fixcols = h->fixcols > 0 ? h->fixcols : (a.p.Np >= 53248 ? 16 : a.p.Np >= 36864 ? 8 : 4);
    a.nsweeps = nsweeps;
    a.sy = h->p.sy;
    a.gbar = (int*)(h->ws + h->L.gbar);
    a.uc = (int*)(h->ws + h->L.uc);
    a.dbg = h->debug ? (long long*)(h->ws + h->L.dbg) : nullptr;
    if (a.dbg) CUDA_TRY(cudaMemsetAsync(a.dbg, 0, kDbgWords * 8, s));
    L.grid = h->pgrid;
    const cudaError_t e = (cudaError_t)fn(L, nullptr);
    if (e != cudaSuccess) return fail(MC_ECUDA, std::string("k_sweep launch: ") + cudaGetErrorString(e));
    return MC_OK;
}

constexpr int64_t kMaxSweepsPerLaunch = 1024;   // keeps a single launch bounded in time

// after a stalled sweep (or before the first one) the scheduling words and the grid barrier must be clean
int reset_scheduling(mc_handle* h) {
    CUDA_TRY(cudaMemsetAsync(h->p.sy, 0, (size_t)h->p.sy_n * 4, h->stream));
    CUDA_TRY(cudaMemsetAsync(h->ws + h->L.gbar, 0, 256, h->stream));
    CUDA_TRY(cudaMemsetAsync(h->ws + h->L.uc, 0, ((size_t)(h->p.Np / 256 + 2) * (kChunkMax / kGroup + 1) + 16) * 4, h->stream));
    return MC_OK;
}

int enqueue_energy(mc_handle* h, double* out_dev, int set_running, int check_overlap) {
    const Params& p = h->p;
    const bool gram = h->form_auto == kFormGram;
    const int rows = (check_overlap || !gram) ? 4 : h->erows;
    const int units = energy_units(p.Np, rows);
    if (check_overlap) k_energy<true, false, 4><<<units, 256, 0, h->stream>>>(p, h->epart);
    else if (!gram) k_energy<false, false, 4><<<units, 256, 0, h->stream>>>(p, h->epart);
    else if (rows == 8) k_energy<false, true, 8><<<units, 256, 0, h->stream>>>(p, h->epart);
    else if (rows == 6) k_energy<false, true, 6><<<units, 256, 0, h->stream>>>(p, h->epart);
    else k_energy<false, true, 4><<<units, 256, 0, h->stream>>>(p, h->epart);
    k_energy_reduce<<<1, 32, 0, h->stream>>>(p, h->epart, units, out_dev, set_running);
    h->launches += 2;
    CUDA_TRY(cudaGetLastError());
    return MC_OK;
}

// Waits for the handle's stream and reports a stalled sweep (the watchdog of persist.cuh): after
// MC_ESTALL the configuration is invalid until mc_set_positions / mc_set_state replaces it.
int sync_and_check(mc_handle* h) {
    int flags[2] = {0, 0};   // DevState::stall, DevState::sched_mismatch (adjacent)
    static_assert(offsetof(DevState, sched_mismatch) == offsetof(DevState, stall) + sizeof(int), "layout");
    CUDA_TRY(cudaMemcpyAsync(flags, &h->p.st->stall, sizeof(flags), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    if (flags[1])
        return fail(MC_ESTALL, "internal error: a sweep's completion counters did not match its plan (" +
                               std::to_string(flags[1]) + " sweeps); the state is not to be trusted");
    if (flags[0])
        return fail(MC_ESTALL, "a sweep stalled (a wait of the sweep kernel exceeded stall_ms); the state is invalid "
                               "until mc_set_positions or mc_set_state replaces it");
    return MC_OK;
}

}  // namespace

extern "C" {

const char* mc_last_error(void) { return g_err.c_str(); }

size_t mc_workspace_bytes(int64_t N) {
    if (N < 1 || N > (int64_t)1 << 30) return 0;
    return make_layout(N).total;
}

int mc_init(mc_handle** out, int64_t N, const double* pos_dev, const double* charges_dev,
            const double* diameters_dev, double cavity_R, double bjerrum_length, double max_disp, uint64_t seed,
            void* workspace_dev, size_t workspace_bytes, void* stream, int validate) {
    if (!out) return fail(MC_EINVAL, "out is null");
    *out = nullptr;
    if (N < 1 || N > (int64_t)1 << 30) return fail(MC_EINVAL, "N out of range");
    if (!pos_dev || !charges_dev || !diameters_dev || !workspace_dev) return fail(MC_EINVAL, "null pointer");
    if (!(cavity_R > 0) || !(bjerrum_length >= 0) || !(max_disp >= 0) || !std::isfinite(cavity_R) ||
        !std::isfinite(bjerrum_length) || !std::isfinite(max_disp))
        return fail(MC_EINVAL, "cavity_R must be > 0, bjerrum_length >= 0, max_disp >= 0, all finite");
    if (cavity_R > 1.0e7) return fail(MC_EINVAL, "cavity_R must not exceed 1e7 (padding particles are parked at 1e9)");
    if (((uintptr_t)workspace_dev % kAlign) != 0) return fail(MC_EINVAL, "workspace must be 256-byte aligned");
    const Layout L = make_layout(N);
    if (workspace_bytes < L.total) return fail(MC_ENOSPACE, "workspace smaller than mc_workspace_bytes(N)");

    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    cudaDeviceProp prop{};
    CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) return fail(MC_ECUDA, "libmcb200 needs an sm_100 device (B200); found sm_" +
                                                    std::to_string(prop.major) + std::to_string(prop.minor));

    mc_handle* h = new mc_handle;
    h->L = L;
    h->ws = (char*)workspace_dev;
    h->stream = (cudaStream_t)stream;
    h->num_sms = prop.multiProcessorCount;
    Params& p = h->p;
    p.N = (int)N; p.Np = padded(N); p.chunk = kChunkMax;
    char* w = h->ws;
    p.xy = (double2*)(w + L.xy); p.zq = (double2*)(w + L.zq); p.hh = (double*)(w + L.hh);
    p.lbq = (double*)(w + L.lbq); p.txy = (double2*)(w + L.txy); p.tz = (double*)(w + L.tz);
    p.lnu = (double*)(w + L.lnu); p.wall = (unsigned char*)(w + L.wall);
    p.Dblk = (double*)(w + L.Dblk); p.OVold = (unsigned*)(w + L.OVold); p.OVnew = (unsigned*)(w + L.OVnew);
    p.log_dE = (double*)(w + L.log_dE); p.log_flags = (unsigned char*)(w + L.log_flags);
    p.st = (DevState*)(w + L.st);
    p.sy = (int*)(w + L.sy);
    p.nn = (double*)(w + L.nn);
    p.S1 = (long long*)(w + L.S1); p.S2 = (long long*)(w + L.S2); p.ovc = (int*)(w + L.ovc);
    p.sy_n = kSyHdr + 4 * (p.Np / 256 + 1);   // header + per-chunk counters
    // measured on B200 (DESIGN.md sections 7 and 9, option sweeps at N = 512 ... 262144): long chunks and wide items pay
    // only when the pair work fills the device; below that the chain paces the sweep and shorter chunks and items keep
    // its inputs ahead of it
    h->prows = p.Np >= 36864 ? 3 : (p.Np >= 512 ? 2 : 1);
    h->pfarcols = p.Np >= 114688 ? 384 : p.Np >= 53248 ? 256 : p.Np >= 36864 ? 128 : 64;
    h->pnear = p.Np >= 36864 ? 4 : 8;
    p.R = cavity_R; p.lB = bjerrum_length; p.max_disp = max_disp; p.seed = seed;
    p.wait_limit_ns = 2000000000ull;
    p.pos_bits = 64;
    h->epart = (double*)(w + L.epart);
    h->centres = (int*)(w + L.centres);
    h->ccount = (int*)(w + L.ccount);
    h->stage_pos = (double*)(w + L.stage_pos);

    auto bail = [&](int code) { delete h; return code; };
    cudaError_t e = cudaMemsetAsync(w, 0, L.total, h->stream);
    if (e != cudaSuccess) return bail(fail(MC_ECUDA, std::string("memset: ") + cudaGetErrorString(e)));
    const int nb = (p.Np + 255) / 256;
    {
        const unsigned long long ones = ~0ull;
        e = cudaMemcpyAsync(&p.st->dmin_bits, &ones, sizeof(ones), cudaMemcpyHostToDevice, h->stream);
        if (e != cudaSuccess) return bail(fail(MC_ECUDA, std::string("init: ") + cudaGetErrorString(e)));
    }
    k_pack<<<nb, 256, 0, h->stream>>>(p, pos_dev, charges_dev, diameters_dev);
    k_check_particles<<<nb, 256, 0, h->stream>>>(p, diameters_dev);
    h->launches += 2;
    if (validate) {
        const int rc = enqueue_energy(h, nullptr, 1, 1);   // exact differences: no geometry assumption yet
        if (rc != MC_OK) return bail(rc);
    }
    DevState st{};
    e = cudaMemcpyAsync(&st, p.st, sizeof(st), cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return bail(fail(MC_ECUDA, std::string("init: ") + cudaGetErrorString(e)));
    h->all_d_equal = st.d_differs == 0;
    h->uniform_d = h->allow_uniform && h->all_d_equal;
    if (st.err != 0) {
        if (st.err <= -1000) return bail(fail(MC_EINVAL, "non-finite input or diameter <= 0"));
        if (st.err == -3) return bail(fail(MC_EOUTSIDE, "an ion sticks out of the cavity"));
        return bail(fail(MC_EOVERLAP, "two ions overlap in the initial configuration"));
    }
    double dmin;
    std::memcpy(&dmin, &st.dmin_bits, sizeof(dmin));
    if (!(dmin > 0) || cavity_R / dmin > 1.0e6)
        return bail(fail(MC_EINVAL, "cavity_R / smallest diameter exceeds 1e6: FP64 positions no longer resolve 1e-10 d"));
    // pair-distance form by geometry (persist.cuh): the cheapest one whose error stays inside the dE bar
    h->form_auto = cavity_R / dmin <= kGramMaxRatio ? kFormGram : max_disp / dmin <= kDiffWMaxRatio ? kFormDiffW : kFormCanon;
    h->form = h->form_auto;
    p.ov_tol = 0x1.0p-20 * dmin * dmin;
    *out = h;
    return MC_OK;
}

int mc_free(mc_handle* h) {
    if (!h) return MC_OK;
    cudaStreamSynchronize(h->stream);
    delete h;
    return MC_OK;
}

int mc_sweep(mc_handle* h, int64_t n) {
    if (!h || n < 0) return fail(MC_EINVAL, "bad handle or n < 0");
    while (n > 0) {
        const int64_t m = std::min(n, kMaxSweepsPerLaunch);
        const int rc = launch_sweep(h, h->stream, (int)m);
        if (rc != MC_OK) return rc;
        h->launches += 1;
        n -= m;
    }
    return MC_OK;
}

int mc_sweep_reduction(mc_handle* h, int64_t n) {
    if (!h || n < 0) return fail(MC_EINVAL, "bad handle or n < 0");
    const Params& p = h->p;
    // the accumulators of the selected particle must be clean (k_sweep leaves its last sweep's sums in them)
    CUDA_TRY(cudaMemsetAsync(p.S1, 0, (size_t)p.Np * 8, h->stream));
    CUDA_TRY(cudaMemsetAsync(p.S2, 0, (size_t)p.Np * 8, h->stream));
    CUDA_TRY(cudaMemsetAsync(p.ovc, 0, (size_t)p.Np * 4, h->stream));
    const int blocks = (p.N + kRedThreads - 1) / kRedThreads;
    for (int64_t s = 0; s < n; ++s) {
        for (int i = 0; i < p.N; ++i) k_reduction_trial<<<blocks, kRedThreads, 0, h->stream>>>(p, i);
        h->launches += (uint64_t)p.N;
        CUDA_TRY(cudaGetLastError());
    }
    return MC_OK;
}

int mc_energy(mc_handle* h, double* E_host) {
    if (!h || !E_host) return fail(MC_EINVAL, "null argument");
    double* out = h->epart + (size_t)energy_units(h->p.Np);
    const int rc = enqueue_energy(h, out, 0, 0);
    if (rc != MC_OK) return rc;
    CUDA_TRY(cudaMemcpyAsync(E_host, out, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    return sync_and_check(h);
}

int mc_energy_dev(mc_handle* h, double* E_dev) {
    if (!h || !E_dev) return fail(MC_EINVAL, "null argument");
    return enqueue_energy(h, E_dev, 0, 0);
}

int mc_sweep_timed(mc_handle* h, int64_t n, double* ms_host) {
    if (!h || !ms_host || n < 1 || n > kMaxSweepsPerLaunch) return fail(MC_EINVAL, "null argument or n outside 1..1024");
    cudaEvent_t ev[2];
    for (auto& x : ev) CUDA_TRY(cudaEventCreate(&x));
    CUDA_TRY(cudaEventRecord(ev[0], h->stream));
    const int rc = launch_sweep(h, h->stream, (int)n);       // the launch of mc_sweep(h, n)
    if (rc != MC_OK) return rc;
    CUDA_TRY(cudaEventRecord(ev[1], h->stream));
    h->launches += 1;
    const int rs = sync_and_check(h);
    float ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&ms, ev[0], ev[1]));
    for (auto& x : ev) cudaEventDestroy(x);
    *ms_host = ms;
    return rs;
}

int mc_pair_hist(mc_handle* h, double bin_width, int nbins, double centre_rmax, uint64_t* hist_dev,
                 uint64_t* n_centres_dev) {
    if (!h || !hist_dev || !n_centres_dev) return fail(MC_EINVAL, "null argument");
    if (!(bin_width > 0) || nbins < 1 || nbins > 8192 || !(centre_rmax >= 0))
        return fail(MC_EINVAL, "bin_width > 0, 1 <= nbins <= 8192, centre_rmax >= 0 required");
    const Params& p = h->p;
    const double inv_w = 1.0 / bin_width;
    const double rcut = (double)nbins * bin_width * (1.0 + 1e-9);
    const double cut2 = rcut * rcut;
    // spatially sorted copy of the configuration (Morton order of cells of about rcut / 2)
    CellGrid g{};
    g.dim = (int)std::min<double>(kCellDim, std::max(1.0, std::floor(2.0 * p.R / (0.5 * rcut))));
    g.lo = -p.R;
    g.inv_edge = (double)g.dim / (2.0 * p.R);
    char* w = h->ws;
    int* code = (int*)(w + h->L.hcode);
    int* ccnt = (int*)(w + h->L.hcount);
    int* ccur = (int*)(w + h->L.hcursor);
    double2* sxy = (double2*)(w + h->L.hsxy);
    double2* szq = (double2*)(w + h->L.hszq);
    double* bbox = (double*)(w + h->L.hbbox);
    const int nb = (p.N + 255) / 256;
    CUDA_TRY(cudaMemsetAsync(ccnt, 0, (size_t)kCells * 4, h->stream));
    CUDA_TRY(cudaMemsetAsync(h->ccount, 0, 4, h->stream));
    k_cell_count<<<nb, 256, 0, h->stream>>>(p, g, code, ccnt);
    k_cell_scan<<<1, 1024, 0, h->stream>>>(ccnt, ccur);
    k_cell_fill<<<nb, 256, 0, h->stream>>>(p, code, ccur, sxy, szq);
    k_tile_bbox<<<nb, 256, 0, h->stream>>>(sxy, szq, p.N, bbox);
    Params ps = p;
    ps.xy = sxy;
    ps.zq = szq;
    k_centres_sorted<<<(p.N + 1023) / 1024, 1024, 0, h->stream>>>(ps, centre_rmax, h->centres, h->ccount,
                                                                 (unsigned long long*)n_centres_dev);
    const size_t smem = (size_t)4 * nbins * sizeof(unsigned);
    if (smem > 32 * 1024)
        CUDA_TRY(cudaFuncSetAttribute(k_hist, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    dim3 grid(nb, h->hist_slices);
    k_hist<<<grid, 256, smem, h->stream>>>(ps, h->centres, h->ccount, bbox, inv_w, nbins, cut2,
                                           (unsigned long long*)hist_dev);
    h->launches += 6;
    CUDA_TRY(cudaGetLastError());
    return MC_OK;
}

int mc_get_positions(mc_handle* h, double* pos_dev_out) {
    if (!h || !pos_dev_out) return fail(MC_EINVAL, "null argument");
    k_unpack<<<(h->p.N + 255) / 256, 256, 0, h->stream>>>(h->p, pos_dev_out);
    h->launches += 1;
    CUDA_TRY(cudaGetLastError());
    return MC_OK;
}

int mc_set_positions(mc_handle* h, const double* pos_dev) {
    if (!h || !pos_dev) return fail(MC_EINVAL, "null argument");
    k_pack<<<(h->p.Np + 255) / 256, 256, 0, h->stream>>>(h->p, pos_dev, nullptr, nullptr);
    k_set_state<<<1, 1, 0, h->stream>>>(h->p.st, 0ull, 0, 0.0, 0);
    h->launches += 2;
    CUDA_TRY(cudaGetLastError());
    const int rc = reset_scheduling(h);
    if (rc != MC_OK) return rc;
    return enqueue_energy(h, nullptr, 1, 0);
}

int mc_set_state(mc_handle* h, const double* pos_dev, uint64_t sweep_index, double E_running) {
    if (!h || !pos_dev) return fail(MC_EINVAL, "null argument");
    if (!std::isfinite(E_running)) return fail(MC_EINVAL, "E_running must be finite");
    k_pack<<<(h->p.Np + 255) / 256, 256, 0, h->stream>>>(h->p, pos_dev, nullptr, nullptr);
    k_set_state<<<1, 1, 0, h->stream>>>(h->p.st, (unsigned long long)sweep_index, 1, E_running, 1);
    h->launches += 2;
    CUDA_TRY(cudaGetLastError());
    return reset_scheduling(h);
}

int mc_get_sweep_index(mc_handle* h, uint64_t* s_host) {
    if (!h || !s_host) return fail(MC_EINVAL, "null argument");
    unsigned long long s = 0;
    CUDA_TRY(cudaMemcpyAsync(&s, &h->p.st->sweep, sizeof(s), cudaMemcpyDeviceToHost, h->stream));
    const int rc = sync_and_check(h);
    *s_host = s;
    return rc;
}

int mc_set_sweep_index(mc_handle* h, uint64_t s) {
    if (!h) return fail(MC_EINVAL, "null handle");
    k_set_sweep<<<1, 1, 0, h->stream>>>(h->p.st, (unsigned long long)s);
    h->launches += 1;
    CUDA_TRY(cudaGetLastError());
    return MC_OK;
}

int mc_get_stats(mc_handle* h, mc_stats* stats_host) {
    if (!h || !stats_host) return fail(MC_EINVAL, "null argument");
    DevState st{};
    CUDA_TRY(cudaMemcpyAsync(&st, h->p.st, sizeof(st), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    stats_host->accepted = st.accepted; stats_host->veto_overlap = st.veto_overlap;
    stats_host->veto_wall = st.veto_wall; stats_host->near_ties = st.near_ties;
    stats_host->E_running = st.E_run;
    if (st.stall || st.sched_mismatch) return sync_and_check(h);
    return MC_OK;
}

int mc_get_trial_log(mc_handle* h, double* dE_dev, uint8_t* flags_dev) {
    if (!h) return fail(MC_EINVAL, "null handle");
    k_copy_log<<<(h->p.N + 255) / 256, 256, 0, h->stream>>>(h->p, dE_dev, flags_dev);
    h->launches += 1;
    CUDA_TRY(cudaGetLastError());
    return MC_OK;
}

int mc_sweep_host(mc_handle* h, int64_t n, const double* pos_in_host, const double* E_running_in,
                  double* pos_out_host, mc_stats* stats_host) {
    if (!h || n < 0) return fail(MC_EINVAL, "bad handle or n < 0");
    const size_t bytes = 3 * (size_t)h->p.N * sizeof(double);
    if (pos_in_host) {
        CUDA_TRY(cudaMemcpyAsync(h->stage_pos, pos_in_host, bytes, cudaMemcpyHostToDevice, h->stream));
        int rc;
        if (E_running_in) {   // the caller vouches for the running energy of this configuration: no O(N^2) pass
            if (!std::isfinite(*E_running_in)) return fail(MC_EINVAL, "E_running_in must be finite");
            k_pack<<<(h->p.Np + 255) / 256, 256, 0, h->stream>>>(h->p, h->stage_pos, nullptr, nullptr);
            k_set_state<<<1, 1, 0, h->stream>>>(h->p.st, 0ull, 0, *E_running_in, 1);
            h->launches += 2;
            rc = cudaGetLastError() == cudaSuccess ? reset_scheduling(h) : fail(MC_ECUDA, "mc_sweep_host: launch failed");
        } else {
            rc = mc_set_positions(h, h->stage_pos);
        }
        if (rc != MC_OK) return rc;
    }
    int rc = mc_sweep(h, n);
    if (rc != MC_OK) return rc;
    if (pos_out_host) {
        rc = mc_get_positions(h, h->stage_pos);
        if (rc != MC_OK) return rc;
        CUDA_TRY(cudaMemcpyAsync(pos_out_host, h->stage_pos, bytes, cudaMemcpyDeviceToHost, h->stream));
    }
    if (stats_host) return mc_get_stats(h, stats_host);
    return sync_and_check(h);
}

int mc_measure_fp64_peak(void* stream, double millis, double* dfma_per_second_host) {
    if (!dfma_per_second_host || !(millis > 0)) return fail(MC_EINVAL, "bad argument");
    cudaStream_t s = (cudaStream_t)stream;
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    cudaDeviceProp prop{};
    CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
    const int blocks = prop.multiProcessorCount * 8;
    cudaEvent_t a, b;
    CUDA_TRY(cudaEventCreate(&a));
    CUDA_TRY(cudaEventCreate(&b));
    int iters = 2000;
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {
        CUDA_TRY(cudaEventRecord(a, s));
        k_dfma_peak<<<blocks, 256, 0, s>>>(nullptr, iters);
        CUDA_TRY(cudaEventRecord(b, s));
        CUDA_TRY(cudaEventSynchronize(b));
        float ms = 0.f;
        CUDA_TRY(cudaEventElapsedTime(&ms, a, b));
        const double ops = (double)blocks * 256.0 * (double)iters * 64.0;
        if (rep > 0 && ms > 0.f) best = std::max(best, ops / (ms * 1e-3));
        if (ms > 0.f && rep == 0) iters = (int)std::min(4.0e6, std::max(2000.0, iters * millis / ms));
    }
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    CUDA_TRY(cudaGetLastError());
    *dfma_per_second_host = best;
    return MC_OK;
}

int mc_set_option(mc_handle* h, const char* key, int64_t value) {
    if (!h || !key) return fail(MC_EINVAL, "null argument");
    if (!std::strcmp(key, "prows")) {
        if (value < 1 || value > 4) return fail(MC_EINVAL, "prows must be 1, 2, 3 or 4");
        h->prows = (int)value;
    } else if (!std::strcmp(key, "far_cols")) {
        if (value < 8 || value > 65536 || value % 8) return fail(MC_EINVAL, "far_cols must be a multiple of 8 in 8..65536");
        h->pfarcols = (int)value;
    } else if (!std::strcmp(key, "pnear")) {
        if (value < 0 || value > 128) return fail(MC_EINVAL, "pnear must be in 0..128");
        h->pnear = (int)value;
    } else if (!std::strcmp(key, "fix_cols")) {
        if (value != 0 && value != 4 && value != 8 && value != 16) return fail(MC_EINVAL, "fix_cols must be 0 (by N), 4, 8 or 16");
        h->fixcols = (int)value;
    } else if (!std::strcmp(key, "diag_split")) {
        if (value != 0 && value != 1 && value != 2 && value != 4 && value != 8) return fail(MC_EINVAL, "diag_split must be 0 (by N), 1, 2, 4 or 8");
        h->dsplit = (int)value;
    } else if (!std::strcmp(key, "max_ctas")) {
        if (value < 0 || value > 4096) return fail(MC_EINVAL, "max_ctas must be in 0..4096 (0: two per SM)");
        h->max_ctas = (int)value;
        h->pgrid_key = -1;
    } else if (!std::strcmp(key, "wave")) {
        h->pwave = value != 0;
    } else if (!std::strcmp(key, "form")) {
        // -1: the form the geometry allows; 0..2: that one or a more exact one (never a less exact one)
        if (value < -1 || value > kFormCanon) return fail(MC_EINVAL, "form must be -1 (automatic), 0, 1 or 2");
        if (value >= 0 && value < h->form_auto && !h->debug)
            return fail(MC_EINVAL, "this geometry needs a more exact pair-distance form than the one requested");
        h->form = value < 0 ? h->form_auto : (int)value;
    } else if (!std::strcmp(key, "position_bits")) {
        if (value != 32 && value != 64) return fail(MC_EINVAL, "position_bits must be 32 or 64");
        h->p.pos_bits = (int)value;
        if (value == 32) {   // round the current configuration; E_running := its from-scratch energy
            k_round_positions<<<(h->p.N + 255) / 256, 256, 0, h->stream>>>(h->p);
            h->launches += 1;
            CUDA_TRY(cudaGetLastError());
            return enqueue_energy(h, nullptr, 1, 0);
        }
    } else if (!std::strcmp(key, "uniform_path")) {
        h->allow_uniform = value != 0;
        h->uniform_d = h->allow_uniform && h->all_d_equal;
    } else if (!std::strcmp(key, "stall_ms")) {
        if (value < 0 || value > 3600000) return fail(MC_EINVAL, "stall_ms must be in 0..3600000 (0: no limit)");
        h->p.wait_limit_ns = (unsigned long long)value * 1000000ull;
    } else if (!std::strcmp(key, "energy_rows")) {
        if (value != 4 && value != 6 && value != 8) return fail(MC_EINVAL, "energy_rows must be 4, 6 or 8");
        h->erows = (int)value;
    } else if (!std::strcmp(key, "hist_slices")) {
        if (value < 1 || value > 64) return fail(MC_EINVAL, "hist_slices must be in 1..64");
        h->hist_slices = (int)value;
    } else if (!std::strcmp(key, "debug")) {
        h->debug = value != 0;
        if (!h->debug) h->pmode = 0;
    } else if (!std::strcmp(key, "probe")) {
        if (value < 0 || value > 2) return fail(MC_EINVAL, "probe must be 0, 1 or 2");
        if (value != 0 && !h->debug) return fail(MC_EINVAL, "probe needs debug = 1 (its sweeps compute nothing meaningful)");
        h->pmode = (int)value;
    } else {
        return fail(MC_EINVAL, std::string("unknown option ") + key);
    }
    return MC_OK;
}

int mc_get_option(mc_handle* h, const char* key, int64_t* value_host) {
    if (!h || !key || !value_host) return fail(MC_EINVAL, "null argument");
    if (!std::strcmp(key, "prows")) *value_host = h->prows;
    else if (!std::strcmp(key, "far_cols")) *value_host = h->pfarcols;
    else if (!std::strcmp(key, "pnear")) *value_host = h->pnear;
    else if (!std::strcmp(key, "wave")) *value_host = h->pwave ? 1 : 0;
    else if (!std::strcmp(key, "max_ctas")) *value_host = h->max_ctas;
    else if (!std::strcmp(key, "diag_split")) *value_host = h->dsplit;
    else if (!std::strcmp(key, "fix_cols")) *value_host = h->fixcols;
    else if (!std::strcmp(key, "form")) *value_host = h->form;
    else if (!std::strcmp(key, "form_auto")) *value_host = h->form_auto;
    else if (!std::strcmp(key, "position_bits")) *value_host = h->p.pos_bits;
    else if (!std::strcmp(key, "uniform_path")) *value_host = h->uniform_d ? 1 : 0;
    else if (!std::strcmp(key, "stall_ms")) *value_host = (int64_t)(h->p.wait_limit_ns / 1000000ull);
    else if (!std::strcmp(key, "hist_slices")) *value_host = h->hist_slices;
    else if (!std::strcmp(key, "energy_rows")) *value_host = h->erows;
    else if (!std::strcmp(key, "debug")) *value_host = h->debug ? 1 : 0;
    else if (!std::strcmp(key, "probe")) *value_host = h->pmode;
    else if (!std::strcmp(key, "grid")) *value_host = h->pgrid;
    else return fail(MC_EINVAL, std::string("unknown option ") + key);
    return MC_OK;
}

int mc_debug_counters(mc_handle* h, int64_t* out16_host) {
    if (!h || !out16_host) return fail(MC_EINVAL, "null argument");
    CUDA_TRY(cudaMemcpyAsync(out16_host, h->ws + h->L.dbg, 16 * 8, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    return MC_OK;
}

int mc_plan_check(int64_t N, int rows_per_thread, int far_cols, int far_workers, int64_t* out4_host) {
    if (N < 1 || N > (int64_t)1 << 30 || !out4_host) return fail(MC_EINVAL, "bad argument");
    if (rows_per_thread < 1 || rows_per_thread > 4) return fail(MC_EINVAL, "rows_per_thread must be 1, 2, 3 or 4");
    if (far_cols < 8 || far_cols % 8 || far_workers < 0) return fail(MC_EINVAL, "far_cols must be a positive multiple of 8, far_workers >= 0");
    const int Np = padded(N), C = 256 * rows_per_thread, nchunks = (Np + C - 1) / C;
    int64_t items = 0, violations = 0, max_item_cols = 0, urgent = 0;
    std::vector<int> cover((size_t)Np / 8);
    for (int c = 0; c < nchunks; ++c) {
        const int row0 = c * C, nrows = chunk_rows(Np, C, c);
        std::fill(cover.begin(), cover.end(), 0);
        auto mark = [&](int col0, int ncol) {
            if (col0 < 0 || ncol <= 0 || col0 % 8 || ncol % 8 || col0 + ncol > Np) { ++violations; return; }
            for (int k = col0 / 8; k < (col0 + ncol) / 8; ++k) ++cover[k];
            max_item_cols = std::max<int64_t>(max_item_cols, ncol);
            ++items;
        };
        // FAR-L and FAR-U items, as the kernel slices them
        for (int pass = 0; pass < 2; ++pass) {
            const int cb = pass == 0 ? 0 : row0 + nrows;
            const int ncols = pass == 0 ? farL_cols(C, c) : farU_cols(Np, C, c);
            const int nf = far_slices(ncols, far_cols, far_workers);
            if ((ncols > 0) != (nf > 0)) ++violations;
            for (int k = 0; k < nf; ++k) {
                const int v0 = slice_bound(ncols, nf, k), v1 = slice_bound(ncols, nf, k + 1);
                mark(cb + v0, v1 - v0);
            }
            if (nf > 0 && slice_bound(ncols, nf, nf) != ncols) ++violations;
        }
        // urgent items: MID (chunk c-2), FIX (chunk c-1)
        if (c >= 2) for (int j = 0; j < C / kMidCols; ++j) { mark(row0 - 2 * C + j * kMidCols, kMidCols); ++urgent; }
        if (c >= 1) for (int j = 0; j < C / kFixCols; ++j) { mark(row0 - C + j * kFixCols, kFixCols); ++urgent; }
        if (urgent_items(C, c) != (c >= 2 ? C / kMidCols : 0) + (c >= 1 ? C / kFixCols : 0)) ++violations;
        // DIAG covers the chunk's own columns
        for (int k = row0 / 8; k < (row0 + nrows) / 8; ++k) ++cover[k];
        items += diag_items(nrows, 1);
        for (int k = 0; k < Np / 8; ++k) violations += cover[k] != 1;
    }
    // the urgent items by release unit, as fetch_item (persist.cuh) hands them out: every (chunk, MID item) and
    // (chunk, FIX item) exactly once, in non-decreasing order of the chain progress that releases them
    for (int fixcols : {4, 8, 16}) {
        const int GPC = C / kGroup, nper = kGroup / fixcols, nmid = C / kMidCols, nfix = C / fixcols;
        std::vector<int> seen((size_t)nchunks * (nmid + nfix), 0);
        int last_need = 0;
        const int units = urgent_units(C, nchunks);
        for (int k = 0; k < units; ++k) {
            int c, g, mid;
            if (k < GPC) { c = 1; g = k; mid = 0; }
            else { c = 2 + (k - GPC) / (GPC + 1); g = (k - GPC) % (GPC + 1) - 1; mid = g < 0 ? 1 : 0; }
            const int need = mid ? (c - 1) * GPC : (c - 1) * GPC + g + 1;
            if (need < last_need || c >= nchunks) ++violations;
            last_need = need;
            for (int v = 0; v < (mid ? nmid : nper); ++v) {
                const int j = mid ? v : g * nper + v;
                if (c < nchunks) ++seen[(size_t)c * (nmid + nfix) + (mid ? j : nmid + j)];
            }
        }
        for (int c = 0; c < nchunks; ++c)
            for (int j = 0; j < nmid + nfix; ++j) {
                const int want = j < nmid ? (c >= 2 ? 1 : 0) : (c >= 1 ? 1 : 0);
                violations += seen[(size_t)c * (nmid + nfix) + j] != want;
            }
    }
    out4_host[0] = items; out4_host[1] = violations; out4_host[2] = max_item_cols; out4_host[3] = urgent;
    return MC_OK;
}

int mc_debug_peek(mc_handle* h, int32_t* out_host, int n) {
    // n > 0: the first n scheduling words (live, then the snapshot); n < 0: the first -n 32-bit words of the diagnostic counters
    if (!h || !out_host || n == 0 || n > 2 * h->p.sy_n || -(int64_t)n * 4 > (int64_t)(kDbgWords * 8))
        return fail(MC_EINVAL, "bad argument");
    cudaStream_t s2;
    CUDA_TRY(cudaStreamCreateWithFlags(&s2, cudaStreamNonBlocking));
    const void* src = n < 0 ? (const void*)(h->ws + h->L.dbg) : (const void*)h->p.sy;
    const cudaError_t e = cudaMemcpyAsync(out_host, src, (size_t)(n < 0 ? -n : n) * 4, cudaMemcpyDeviceToHost, s2);
    const cudaError_t e2 = cudaStreamSynchronize(s2);
    cudaStreamDestroy(s2);
    if (e != cudaSuccess || e2 != cudaSuccess) return fail(MC_ECUDA, "mc_debug_peek: copy failed");
    return MC_OK;
}

int mc_get_launch_count(mc_handle* h, uint64_t* n_host) {
    if (!h || !n_host) return fail(MC_EINVAL, "null argument");
    *n_host = h->launches;
    return MC_OK;
}

}  // extern "C"

// =============================================================================================
// mc_energy_noalloc: the from-scratch energy (a5) for callers that cannot allocate device memory
// (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  No handle,
// no workspace: the per-CTA partial sums live in a file-scope __device__ array that every GPU loading
// this library holds until exit.  Same decomposition and summation order as k_energy (aux_kernels.cuh)
// with exact coordinate differences (reading G11), on the caller's raw arrays.
// =============================================================================================
namespace {

// 1024 x 256 units of the upper triangle at N = MC_NOALLOC_MAX_N: sum_{rb < 128} (512 - 4 rb) = 33,024 partials
constexpr int kNoAllocMaxUnits = 33024;
static_assert(MC_NOALLOC_MAX_N % 1024 == 0, "the unit count below assumes whole row blocks");
static_assert((MC_NOALLOC_MAX_N / 1024) * (MC_NOALLOC_MAX_N / 256) -
                      4 * ((MC_NOALLOC_MAX_N / 1024 - 1) * (MC_NOALLOC_MAX_N / 1024) / 2) == kNoAllocMaxUnits, "unit count");
static __device__ __align__(256) double g_noalloc_scratch[kNoAllocMaxUnits];   // 264,192 bytes per GPU

// one unit = rows [rb 1024, rb 1024 + 1024) x columns [j0, j0 + 256), pairs j > i only; 4 rows per thread
__global__ void __launch_bounds__(256, 2) k_energy_raw(const double* __restrict__ pos, const double* __restrict__ chg,
                                                       int N, double* __restrict__ part) {
    constexpr int kRows = 4, kBlock = 256 * kRows;
    __shared__ double sx[kETile], sy[kETile], sz[kETile], sq[kETile];
    __shared__ double red[8];
    const int tid = threadIdx.x;
    int unit = blockIdx.x, rb = 0;
    for (;;) {
        const int n = ((N - rb * kBlock) + kETile - 1) / kETile;
        if (unit < n) break;
        unit -= n;
        ++rb;
    }
    const int j0 = rb * kBlock + unit * kETile;
    const int cnt = min(kETile, N - j0);
    double x[kRows], y[kRows], z[kRows], q[kRows], acc[kRows];
#pragma unroll
    for (int u = 0; u < kRows; ++u) {
        const int i = rb * kBlock + u * 256 + tid;
        const bool live = i < N;
        x[u] = live ? pos[i] : 0.0; y[u] = live ? pos[(size_t)N + i] : 0.0; z[u] = live ? pos[2 * (size_t)N + i] : 0.0;
        q[u] = live ? chg[i] : 0.0;
        acc[u] = 0.0;
    }
    if (tid < cnt) {
        sx[tid] = pos[j0 + tid]; sy[tid] = pos[(size_t)N + j0 + tid]; sz[tid] = pos[2 * (size_t)N + j0 + tid];
        sq[tid] = chg[j0 + tid];
    }
    __syncthreads();
    const bool diagonal = unit < kBlock / kETile;
    if (!diagonal) {
#pragma unroll 2
        for (int j = 0; j < cnt; ++j) {
            const double ax = sx[j], ay = sy[j], az = sz[j], aq = sq[j];
#pragma unroll
            for (int u = 0; u < kRows; ++u) {
                const double r2 = dist2(__dadd_rn(x[u], -ax), __dadd_rn(y[u], -ay), __dadd_rn(z[u], -az));
                acc[u] = __fma_rn(aq, rsqrt_fast(r2), acc[u]);
            }
        }
    } else {
        for (int j = 0; j < cnt; ++j) {
            const double ax = sx[j], ay = sy[j], az = sz[j], aq = sq[j];
#pragma unroll
            for (int u = 0; u < kRows; ++u) {
                const int i = rb * kBlock + u * 256 + tid;
                if (j0 + j > i && i < N) {
                    const double r2 = dist2(__dadd_rn(x[u], -ax), __dadd_rn(y[u], -ay), __dadd_rn(z[u], -az));
                    acc[u] = __fma_rn(aq, rsqrt_fast(r2), acc[u]);
                }
            }
        }
    }
    // off the diagonal a dead row (i >= N) sits at the origin with q = 0: its sum is finite unless an ion sits exactly
    // there, so it is dropped explicitly rather than multiplied by zero
    double v = 0.0;
#pragma unroll
    for (int u = 0; u < kRows; ++u) {
        const int i = rb * kBlock + u * 256 + tid;
        if (i < N) v = __dadd_rn(v, __dmul_rn(q[u], acc[u]));
    }
    v = warp_sum(v);
    if ((tid & 31) == 0) red[tid >> 5] = v;
    __syncthreads();
    if (tid == 0) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t = __dadd_rn(t, red[w]);
        part[blockIdx.x] = t;
    }
}

// *out = l_B * sum of the partials in index order (one warp)
__global__ void __launch_bounds__(32) k_energy_raw_reduce(const double* __restrict__ part, int nparts, double lB, double* out) {
    double acc = 0.0;
    for (int k = threadIdx.x; k < nparts; k += 32) acc = __dadd_rn(acc, part[k]);
    acc = warp_sum(acc);
    if (threadIdx.x == 0) *out = __dmul_rn(lB, acc);
}

// device address of g_noalloc_scratch, looked up once per device with that device current (in host code the array's
// name is a host-side stand-in, not a device address)
constexpr int kNoAllocMaxDevices = 64;
double* g_noalloc_ptr[kNoAllocMaxDevices] = {};
std::mutex g_noalloc_mutex;

}  // namespace

extern "C" int mc_energy_noalloc(int64_t N, const double* pos_dev, const double* charges_dev, double bjerrum_length,
                                 double* E_dev, void* stream) {
    if (!pos_dev || !charges_dev || !E_dev) return fail(MC_EINVAL, "mc_energy_noalloc: null argument");
    if (N < 1 || N > MC_NOALLOC_MAX_N)
        return fail(MC_ENOSPACE, "mc_energy_noalloc: N = " + std::to_string(N) + " is outside 1.." +
                                     std::to_string(MC_NOALLOC_MAX_N) + " (MC_NOALLOC_MAX_N: the size the static scratch "
                                     "array is built for); use mc_init + mc_energy for larger systems");
    if (!std::isfinite(bjerrum_length)) return fail(MC_EINVAL, "mc_energy_noalloc: bjerrum_length must be finite");
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kNoAllocMaxDevices) return fail(MC_EINVAL, "mc_energy_noalloc: device ordinal beyond 63");
    double* scratch = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_noalloc_mutex);
        if (!g_noalloc_ptr[dev]) {
            double* ptr = nullptr;
            const cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch);
            if (e != cudaSuccess || !ptr)
                return fail(MC_ECUDA, std::string("mc_energy_noalloc: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
            g_noalloc_ptr[dev] = ptr;
        }
        scratch = g_noalloc_ptr[dev];
    }
    const int units = energy_units((int)N, 4);
    if (units > kNoAllocMaxUnits) return fail(MC_ENOSPACE, "mc_energy_noalloc: internal: unit count beyond the scratch array");
    cudaStream_t st = (cudaStream_t)stream;
    // every partial a call reads is written by that call first: nothing in the array has to start at zero
    k_energy_raw<<<units, 256, 0, st>>>(pos_dev, charges_dev, (int)N, scratch);
    k_energy_raw_reduce<<<1, 32, 0, st>>>(scratch, units, bjerrum_length, E_dev);
    CUDA_TRY(cudaGetLastError());
    return MC_OK;
}
