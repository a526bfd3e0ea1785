// oracle/oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU statement of what the hot path of
// arXiv 1602.05716 computes: the exact sequential-order Metropolis sweep of a
// primitive-model electrolyte (charged hard spheres, bare 1/r Coulomb, hard-wall
// spherical cavity).  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may load this.  It shares no code with
// paper_1602_05716_b200/csrc (the CUDA path) and neither includes the other.
//
// Citations are PAPER.md:<line> (+ section / equation / algorithm) and the
// readings G1..G19 of SURVEY.md section 8(c), repeated in DESIGN.md.
//
//   step = select / trial / accept            PAPER.md:43-50  (Sec. 2, Eq. 1)
//   sequential updating, ascending order
//   dE_ij uses x'_j for j<i, x_j for j>i       PAPER.md:60-63  (Eq. 2)
//   all energy arithmetic in FP64              PAPER.md:99     (Sec. 3.3)
//   overlap is a separate indicator
//   accept iff u < exp(-dE), strict            PAPER.md:201, 225 (Alg. 4)
//   hard-wall spherical domain                 PAPER.md:351    (Sec. 5.2)
//   g(r) from bulk centres only
//
// Pins (tests/test_oracle_*.py): Philox known answers, uniform mapping,
// two-ion closed form, brute-force total-energy differences on tiny N,
// energy bookkeeping invariant, hard constraints, degenerate cases, two- and
// three-ion Boltzmann laws by quadrature, re-entrancy.  Nothing here is
// "parity unpinned".
//
// Build: g++ -O3 -mavx2 -mfma -ffp-contract=off -fopenmp -shared -fPIC

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

#define ORACLE_OK 0
#define ORACLE_EINVAL (-1)
#define ORACLE_EOVERLAP (-2)
#define ORACLE_EOUTSIDE (-3)

namespace {

// ---------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), written from the round
// description (reading G9): 10 rounds; before every round but the first the key
// is bumped by the Weyl constants; a round maps
//   (c0,c1,c2,c3) -> (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)).
// ---------------------------------------------------------------------------
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) {
            k0 += 0x9E3779B9u;
            k1 += 0xBB67AE85u;
        }
        const uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        const uint32_t h0 = (uint32_t)(p0 >> 32), l0 = (uint32_t)p0;
        const uint32_t h1 = (uint32_t)(p1 >> 32), l1 = (uint32_t)p1;
        const uint32_t n0 = h1 ^ c1 ^ k0;
        const uint32_t n1 = l1;
        const uint32_t n2 = h0 ^ c3 ^ k1;
        const uint32_t n3 = l0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Reading G10: u = (2k+1) * 2^-53 with k = top 52 bits of the 64-bit word
// (hi<<32)|lo.  u lies in (0,1), is exactly representable, and so is u - 1/2.
double uniform_open01(uint32_t lo, uint32_t hi) {
    const uint64_t w = ((uint64_t)hi << 32) | (uint64_t)lo;
    const uint64_t k = w >> 12;
    return (double)(2 * k + 1) * 0x1.0p-53;
}

struct Handle {
    int64_t N = 0;
    std::vector<double> x, y, z, q, d;
    double R = 0, lB = 0, max_disp = 0;
    uint64_t seed = 0, sweep = 0;
    int threads = 1;
    // 64: positions are FP64 (north star, reading G8).  32: the paper's storage format -- every position the
    // chain holds is an FP32 value (float4 X_dev); all arithmetic on them stays FP64.
    int pos_bits = 64;
    // statistics since init
    uint64_t n_accept = 0, n_veto_overlap = 0, n_veto_wall = 0, n_near_tie = 0;
    double E_run = 0;
    // log of the last sweep
    std::vector<double> log_dE, log_scale, log_t;
    std::vector<uint8_t> log_flags;
    std::vector<double> tx, ty, tz;  // trial positions of the last sweep
};

struct Trial {
    double tx, ty, tz, u_acc;
    bool wall_veto;
};

// Alg. 1 with the old position added (reading G1), D = 2*max_disp
// (G2), the explicit fused form fma(u - 1/2, D, x) (G11) and the hard wall
// "sphere wholly inside, touching allowed" (G6).
Trial make_trial(const Handle& h, int64_t i) {
    const uint32_t key[2] = {(uint32_t)h.seed, (uint32_t)(h.seed >> 32)};
    const uint32_t ca[4] = {(uint32_t)i, (uint32_t)h.sweep, (uint32_t)(h.sweep >> 32), 0u};
    const uint32_t cb[4] = {(uint32_t)i, (uint32_t)h.sweep, (uint32_t)(h.sweep >> 32), 1u};
    uint32_t A[4], B[4];
    philox4x32_10(ca, key, A);
    philox4x32_10(cb, key, B);
    const double ux = uniform_open01(A[0], A[1]);
    const double uy = uniform_open01(A[2], A[3]);
    const double uz = uniform_open01(B[0], B[1]);
    Trial t;
    t.u_acc = uniform_open01(B[2], B[3]);
    const double D = 2.0 * h.max_disp;
    t.tx = std::fma(ux - 0.5, D, h.x[i]);
    t.ty = std::fma(uy - 0.5, D, h.y[i]);
    t.tz = std::fma(uz - 0.5, D, h.z[i]);
    if (h.pos_bits == 32) {   // the proposed position is stored as FP32: one more rounding, to nearest
        t.tx = (double)(float)t.tx; t.ty = (double)(float)t.ty; t.tz = (double)(float)t.tz;
    }
    const double a = h.R - 0.5 * h.d[i];
    const double rr = std::fma(t.tz, t.tz, std::fma(t.ty, t.ty, t.tx * t.tx));
    t.wall_veto = rr > a * a;
    return t;
}

// One Metropolis step for particle i against the positions as they are NOW:
// j < i already carry this sweep's decision, j > i not yet (Eq. 2).
// No early exit on overlap.
void metropolis_step(Handle& h, int64_t i) {
    const Trial t = make_trial(h, i);
    const double xi = h.x[i], yi = h.y[i], zi = h.z[i], di = h.d[i];
    const int64_t N = h.N;
    double acc = 0.0, mag = 0.0;
    int64_t ov = 0;
    if (h.threads <= 1) {
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            const double dxo = xi - h.x[j], dyo = yi - h.y[j], dzo = zi - h.z[j];
            const double dxn = t.tx - h.x[j], dyn = t.ty - h.y[j], dzn = t.tz - h.z[j];
            const double r2o = std::fma(dzo, dzo, std::fma(dyo, dyo, dxo * dxo));
            const double r2n = std::fma(dzn, dzn, std::fma(dyn, dyn, dxn * dxn));
            const double sij = 0.5 * (di + h.d[j]);
            ov += (r2n < sij * sij);                       // reading G7: strict, contact allowed
            const double du = 1.0 / std::sqrt(r2n) - 1.0 / std::sqrt(r2o);
            acc += h.q[j] * du;
            mag += std::fabs(h.q[j]) * std::fabs(du);
        }
    } else {
        // Same terms, summed per thread over a static partition of j and then
        // combined; differs from the serial sum by rounding order only.  Used
        // for the large parity cases and the all-core timing.
#pragma omp parallel for schedule(static) reduction(+ : acc, mag, ov) num_threads(h.threads)
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            const double dxo = xi - h.x[j], dyo = yi - h.y[j], dzo = zi - h.z[j];
            const double dxn = t.tx - h.x[j], dyn = t.ty - h.y[j], dzn = t.tz - h.z[j];
            const double r2o = std::fma(dzo, dzo, std::fma(dyo, dyo, dxo * dxo));
            const double r2n = std::fma(dzn, dzn, std::fma(dyn, dyn, dxn * dxn));
            const double sij = 0.5 * (di + h.d[j]);
            ov += (r2n < sij * sij);
            const double du = 1.0 / std::sqrt(r2n) - 1.0 / std::sqrt(r2o);
            acc += h.q[j] * du;
            mag += std::fabs(h.q[j]) * std::fabs(du);
        }
    }
    // energies in k_B T: dE = l_B q_i sum_j q_j (1/r_new - 1/r_old)   (reading G3)
    const double dE = h.lB * h.q[i] * acc;
    const double tt = dE + std::log(t.u_acc);          // accept iff u < exp(-dE), in log form
    const bool clear = !t.wall_veto && ov == 0;
    const bool accept = clear && (tt < 0.0);            // strict (G4)
    const bool near_tie = clear && (std::fabs(tt) < 1e-8);
    h.log_dE[i] = dE;
    h.log_scale[i] = h.lB * std::fabs(h.q[i]) * mag;   // natural scale M_i (G13)
    h.log_t[i] = tt;
    h.log_flags[i] = (uint8_t)((accept ? 1 : 0) | (ov > 0 ? 2 : 0) | (t.wall_veto ? 4 : 0) |
                               (near_tie ? 8 : 0));
    h.tx[i] = t.tx; h.ty[i] = t.ty; h.tz[i] = t.tz;
    if (ov > 0) h.n_veto_overlap++;
    if (t.wall_veto) h.n_veto_wall++;
    if (near_tie) h.n_near_tie++;
    if (accept) {
        h.x[i] = t.tx; h.y[i] = t.ty; h.z[i] = t.tz;    // Eq. 1
        h.E_run += dE;
        h.n_accept++;
    }
}

// E = l_B sum_{i<j} q_i q_j / r_ij in k_B T, ascending loops.
double total_energy(const Handle& h) {
    double E = 0.0;
    for (int64_t i = 0; i < h.N; ++i) {
        for (int64_t j = i + 1; j < h.N; ++j) {
            const double dx = h.x[i] - h.x[j], dy = h.y[i] - h.y[j], dz = h.z[i] - h.z[j];
            const double r2 = std::fma(dz, dz, std::fma(dy, dy, dx * dx));
            E += h.q[i] * h.q[j] / std::sqrt(r2);
        }
    }
    return h.lB * E;
}

int validate(const Handle& h) {
    if (h.N < 1 || !(h.R > 0) || !(h.lB >= 0) || !(h.max_disp >= 0)) return ORACLE_EINVAL;
    if (!std::isfinite(h.R) || !std::isfinite(h.lB) || !std::isfinite(h.max_disp)) return ORACLE_EINVAL;
    for (int64_t i = 0; i < h.N; ++i) {
        if (!std::isfinite(h.x[i]) || !std::isfinite(h.y[i]) || !std::isfinite(h.z[i]) ||
            !std::isfinite(h.q[i]) || !std::isfinite(h.d[i]) || !(h.d[i] > 0))
            return ORACLE_EINVAL;
    }
    for (int64_t i = 0; i < h.N; ++i) {
        const double a = h.R - 0.5 * h.d[i];
        const double rr = std::fma(h.z[i], h.z[i], std::fma(h.y[i], h.y[i], h.x[i] * h.x[i]));
        if (!(a >= 0) || rr > a * a) return ORACLE_EOUTSIDE;
    }
    for (int64_t i = 0; i < h.N; ++i) {
        for (int64_t j = i + 1; j < h.N; ++j) {
            const double dx = h.x[i] - h.x[j], dy = h.y[i] - h.y[j], dz = h.z[i] - h.z[j];
            const double r2 = std::fma(dz, dz, std::fma(dy, dy, dx * dx));
            const double sij = 0.5 * (h.d[i] + h.d[j]);
            if (r2 < sij * sij) return ORACLE_EOVERLAP;
        }
    }
    return ORACLE_OK;
}

}  // namespace

extern "C" {

struct oracle_stats {
    uint64_t accepted, veto_overlap, veto_wall, near_ties;
    double E_running;
};

void oracle_philox4x32_10(const uint32_t* ctr4, const uint32_t* key2, uint32_t* out4) {
    philox4x32_10(ctr4, key2, out4);
}

double oracle_uniform_open01(uint32_t lo, uint32_t hi) { return uniform_open01(lo, hi); }

// pos is SoA [3][N] (x then y then z), host memory; copied.
int oracle_init(void** out, int64_t N, const double* pos, const double* charges,
                const double* diameters, double cavity_R, double bjerrum_length, double max_disp,
                uint64_t seed, int validate_input) {
    if (!out || !pos || !charges || !diameters || N < 1) return ORACLE_EINVAL;
    Handle* h = new Handle;
    h->N = N;
    h->x.assign(pos, pos + N);
    h->y.assign(pos + N, pos + 2 * N);
    h->z.assign(pos + 2 * N, pos + 3 * N);
    h->q.assign(charges, charges + N);
    h->d.assign(diameters, diameters + N);
    h->R = cavity_R; h->lB = bjerrum_length; h->max_disp = max_disp; h->seed = seed;
    h->log_dE.assign(N, 0.0); h->log_scale.assign(N, 0.0); h->log_t.assign(N, 0.0);
    h->log_flags.assign(N, 0);
    h->tx.assign(N, 0.0); h->ty.assign(N, 0.0); h->tz.assign(N, 0.0);
    if (validate_input) {
        const int rc = validate(*h);
        if (rc != ORACLE_OK) { delete h; return rc; }
        h->E_run = total_energy(*h);
    }
    *out = h;
    return ORACLE_OK;
}

void oracle_free(void* hp) { delete (Handle*)hp; }

int oracle_set_threads(void* hp, int n) {
    if (!hp || n < 1) return ORACLE_EINVAL;
    ((Handle*)hp)->threads = n;
    return ORACLE_OK;
}

// Position storage precision: bits = 32 rounds the current positions to
// FP32 (to nearest) and makes every later trial position an FP32 value; E_running is recomputed from scratch.
// bits = 64 only switches the rounding of later trials off.
int oracle_set_position_bits(void* hp, int bits) {
    if (!hp || (bits != 32 && bits != 64)) return ORACLE_EINVAL;
    Handle& h = *(Handle*)hp;
    h.pos_bits = bits;
    if (bits == 32) {
        for (int64_t i = 0; i < h.N; ++i) {
            h.x[i] = (double)(float)h.x[i]; h.y[i] = (double)(float)h.y[i]; h.z[i] = (double)(float)h.z[i];
        }
        h.E_run = total_energy(h);
    }
    return ORACLE_OK;
}

// n full sweeps: particles 0..N-1 in ascending order, exactly once each.
int oracle_sweep(void* hp, int64_t n) {
    if (!hp || n < 0) return ORACLE_EINVAL;
    Handle& h = *(Handle*)hp;
    for (int64_t s = 0; s < n; ++s) {
        for (int64_t i = 0; i < h.N; ++i) metropolis_step(h, i);
        h.sweep += 1;
    }
    return ORACLE_OK;
}

// Trials first..first+count-1 of the CURRENT sweep, without advancing the sweep
// index.  For bounded timing samples and for step-by-step brute-force pins.
int oracle_partial_sweep(void* hp, int64_t first, int64_t count) {
    if (!hp || first < 0 || count < 0) return ORACLE_EINVAL;
    Handle& h = *(Handle*)hp;
    if (first + count > h.N) return ORACLE_EINVAL;
    for (int64_t i = first; i < first + count; ++i) metropolis_step(h, i);
    return ORACLE_OK;
}

int oracle_energy(void* hp, double* E) {
    if (!hp || !E) return ORACLE_EINVAL;
    *E = total_energy(*(Handle*)hp);
    return ORACLE_OK;
}

// hist [2][2][nbins] and n_centres [2] are accumulators (added to).  Species 0 if
// q > 0 else 1.  Ordered pairs (centre i in the bulk, any partner j != i).
// With more than one thread (oracle_set_threads) the centres are shared out over
// threads, each counting into a private copy that is added at the end: integer
// counts, so the result is the serial one whatever the order (reading G17).
int oracle_pair_hist(void* hp, double bin_width, int nbins, double centre_rmax, uint64_t* hist,
                     uint64_t* n_centres) {
    if (!hp || !hist || !n_centres || !(bin_width > 0) || nbins < 1) return ORACLE_EINVAL;
    const Handle& h = *(Handle*)hp;
    const double inv_w = 1.0 / bin_width;
    const double c2 = centre_rmax * centre_rmax;
    // all partners of one centre, counted into hs / ns
    auto centre = [&](int64_t i, uint64_t* hs, uint64_t* ns) {
        const double rr = std::fma(h.z[i], h.z[i], std::fma(h.y[i], h.y[i], h.x[i] * h.x[i]));
        if (!(rr <= c2)) return;
        const int si = h.q[i] > 0 ? 0 : 1;
        ns[si] += 1;
        for (int64_t j = 0; j < h.N; ++j) {
            if (j == i) continue;
            const double dx = h.x[i] - h.x[j], dy = h.y[i] - h.y[j], dz = h.z[i] - h.z[j];
            const double r2 = std::fma(dz, dz, std::fma(dy, dy, dx * dx));
            const double r = std::sqrt(r2);
            const double fb = std::floor(r * inv_w);
            if (fb < (double)nbins) {
                const int sj = h.q[j] > 0 ? 0 : 1;
                hs[((size_t)si * 2 + sj) * (size_t)nbins + (size_t)fb] += 1;
            }
        }
    };
    if (h.threads <= 1) {
        for (int64_t i = 0; i < h.N; ++i) centre(i, hist, n_centres);
    } else {
#pragma omp parallel num_threads(h.threads)
        {
            std::vector<uint64_t> hs((size_t)4 * nbins, 0);
            uint64_t ns[2] = {0, 0};
#pragma omp for schedule(dynamic, 64)
            for (int64_t i = 0; i < h.N; ++i) centre(i, hs.data(), ns);
#pragma omp critical
            {
                for (size_t k = 0; k < hs.size(); ++k) hist[k] += hs[k];
                n_centres[0] += ns[0];
                n_centres[1] += ns[1];
            }
        }
    }
    return ORACLE_OK;
}

int oracle_get_positions(void* hp, double* pos) {
    if (!hp || !pos) return ORACLE_EINVAL;
    const Handle& h = *(Handle*)hp;
    std::memcpy(pos, h.x.data(), sizeof(double) * h.N);
    std::memcpy(pos + h.N, h.y.data(), sizeof(double) * h.N);
    std::memcpy(pos + 2 * h.N, h.z.data(), sizeof(double) * h.N);
    return ORACLE_OK;
}

int oracle_set_positions(void* hp, const double* pos) {
    if (!hp || !pos) return ORACLE_EINVAL;
    Handle& h = *(Handle*)hp;
    h.x.assign(pos, pos + h.N);
    h.y.assign(pos + h.N, pos + 2 * h.N);
    h.z.assign(pos + 2 * h.N, pos + 3 * h.N);
    return ORACLE_OK;
}

int oracle_get_sweep_index(void* hp, uint64_t* s) {
    if (!hp || !s) return ORACLE_EINVAL;
    *s = ((Handle*)hp)->sweep;
    return ORACLE_OK;
}

int oracle_set_sweep_index(void* hp, uint64_t s) {
    if (!hp) return ORACLE_EINVAL;
    ((Handle*)hp)->sweep = s;
    return ORACLE_OK;
}

int oracle_get_stats(void* hp, oracle_stats* st) {
    if (!hp || !st) return ORACLE_EINVAL;
    const Handle& h = *(Handle*)hp;
    st->accepted = h.n_accept; st->veto_overlap = h.n_veto_overlap; st->veto_wall = h.n_veto_wall;
    st->near_ties = h.n_near_tie; st->E_running = h.E_run;
    return ORACLE_OK;
}

// Log of the last sweep (or of the trials run by oracle_partial_sweep):
// dE [N] in k_BT; flags [N]: bit0 accept, bit1 overlap veto, bit2 wall veto,
// bit3 near-tie; scale [N] = M_i of reading G13; t [N] = dE + ln u;
// trial [3][N] = proposed positions.  Any pointer may be null.
int oracle_get_trial_log(void* hp, double* dE, uint8_t* flags, double* scale, double* t,
                         double* trial) {
    if (!hp) return ORACLE_EINVAL;
    const Handle& h = *(Handle*)hp;
    if (dE) std::memcpy(dE, h.log_dE.data(), sizeof(double) * h.N);
    if (flags) std::memcpy(flags, h.log_flags.data(), h.N);
    if (scale) std::memcpy(scale, h.log_scale.data(), sizeof(double) * h.N);
    if (t) std::memcpy(t, h.log_t.data(), sizeof(double) * h.N);
    if (trial) {
        std::memcpy(trial, h.tx.data(), sizeof(double) * h.N);
        std::memcpy(trial + h.N, h.ty.data(), sizeof(double) * h.N);
        std::memcpy(trial + 2 * h.N, h.tz.data(), sizeof(double) * h.N);
    }
    return ORACLE_OK;
}

}  // extern "C"
