// xy_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU implementation of one Monte Carlo step (MCS) of the
// 3-D classical XY model over R parallel-tempering replicas, written from the text of
// arXiv:1211.0780 (PAPER.md, cited below as P:<line>) and the readings frozen in DESIGN.md
// ("Readings of the paper").  It exists so that tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs can check and time the CUDA path against
// something that can be verified against the paper by eye.  Nothing else may import, link
// or call it.  It shares no code, header, table or constant generator with
// paper_1211_0780_b200/csrc/ (the CUDA path); it has its own Philox4x32-10.
//
// Arithmetic: angles are STORED as fp32 (so a state is exchangeable bit-for-bit with the
// GPU), every computation is done in double with libm, in the paper's order, without
// blocking, fusion, caching of sin/cos, or reordering.  One thread per replica slot at most
// (replicas are independent within a sweep; the RNG is counter-based, so the result does
// not depend on the thread count).
//
// What pins it (tests/test_oracle_pins.py, none of which re-types these formulas):
//   Philox4x32-10      known-answer vectors (tests/golden/philox4x32_10_kat.txt)
//   init / Metropolis  beta=0: every proposal accepted, state predictable from Philox alone;
//                      high-temperature series <cos> = t + 8 t^3 t' (t = I1/I0);
//                      L=2 exact <E> from a brute-force 7-D quadrature; T=0 fixed point
//   over-relaxation    energy conservation, involution, helical-state fixed point
//   measure            ordered / helical / staggered closed forms, global-rotation invariance,
//                      brute-force bond loop in Python
//   PT exchange        equal-beta forced swaps (known permutation), R=1 no-op,
//                      <E> invariance with PT on/off
//   stiffness sums     ordered and helical closed forms per axis, E = -(Cx+Cy+Cz), odd / even
//                      under theta -> -theta, global-rotation invariance, brute-force bond loop in Python
// Parity unpinned: nothing in this file.
//
// Build: g++ -O2 -std=c++17 -shared -fPIC -pthread xy_oracle.cpp -o libxy_oracle.so
// (no -ffast-math: libm double semantics are part of the definition).

#include <cmath>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>

namespace {

// ---------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  BASELINE.json north_star: "the
// Philox4x32-10 counter-based RNG, keyed by (seed, replica, site, sweep, stream-id)".
// Replaces the paper's Warp Generator, which is not available.
// ---------------------------------------------------------------------------------------
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;   // round multipliers
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;   // Weyl key increments
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += W0; k1 += W1; }
        const uint64_t p0 = (uint64_t)M0 * c0;
        const uint64_t p1 = (uint64_t)M1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n1 = (uint32_t)p1;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        const uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Stream ids (counter word 3).  DESIGN.md reading R12: the two Metropolis colour passes of
// one sweep use DIFFERENT streams, so that a black site and the white site next to it never
// see the same random numbers.
enum : uint32_t { STREAM_INIT = 0, STREAM_MET_BLACK = 1, STREAM_MET_WHITE = 2, STREAM_PT = 3 };

const float  TWO_PI_F = 6.2831855f;            // 0x40C90FDB, fp32 nearest to 2*pi
const double TWO_PI_D = 6.283185307179586476925286766559;

// u24(w): top 24 bits of a word as a fraction in [0,1); exact in fp32.
inline float u24(uint32_t w) { return (float)(w >> 8) * (1.0f / 16777216.0f); }

struct Ctx {
    int L = 0, R = 0;
    int64_t N = 0;
    uint64_t seed = 0;
    std::vector<double> betas;          // by rank k (the caller's array)          [P:45]
    std::vector<double> beta_of_slot;   // current beta label of each spin array   [reading R11]
    std::vector<int> slot_at_rank;      // which spin array holds rank k
    std::vector<float> theta;           // [R][z][y][x], x fastest, fp32 storage   [P:62]
    uint32_t n_met = 0, n_or = 0, n_pt = 0;
    int n_threads = 1;
    std::vector<int> active;            // slots that sweeps/measure touch (default: all)
    std::vector<uint64_t> met_acc;      // accepted Metropolis proposals per slot
    std::vector<uint64_t> pt_acc;       // accepted swaps per pair (k,k+1)
    // optional traces (caller-owned, may be null)
    double* tr_met_p = nullptr;         // [R][N] acceptance probability exp(-beta dE)
    float*  tr_met_u = nullptr;         // [R][N] the uniform it was compared with
    double* tr_or_h = nullptr;          // [R][N] |h_i| seen by the over-relaxation update
    double* tr_pt_p = nullptr;          // [R-1]  swap probability (unclamped) per pair; NaN if not attempted
    double* tr_pt_u = nullptr;          // [R-1]  the uniform
};

inline int wrap(int a, int L) { return a < 0 ? a + L : (a >= L ? a - L : a); }

// Local field h_i = (sum_j cos theta_j, sum_j sin theta_j) over the six nearest neighbours
// with periodic boundaries [P:23-28 Eq. 1; P:38 H_i up to the sign, reading R5].  For L=2
// the +mu and -mu neighbours coincide and are both counted.
inline void local_field(const Ctx& c, const float* th, int x, int y, int z, double& hx, double& hy) {
    const int L = c.L;
    const int xs[2] = { wrap(x - 1, L), wrap(x + 1, L) };
    const int ys[2] = { wrap(y - 1, L), wrap(y + 1, L) };
    const int zs[2] = { wrap(z - 1, L), wrap(z + 1, L) };
    hx = 0.0; hy = 0.0;
    for (int s = 0; s < 2; ++s) {
        const double tx = (double)th[xs[s] + (int64_t)L * (y + (int64_t)L * z)];
        const double ty = (double)th[x + (int64_t)L * (ys[s] + (int64_t)L * z)];
        const double tz = (double)th[x + (int64_t)L * (y + (int64_t)L * zs[s])];
        hx += std::cos(tx); hy += std::sin(tx);
        hx += std::cos(ty); hy += std::sin(ty);
        hx += std::cos(tz); hy += std::sin(tz);
    }
}

// One Metropolis colour pass over one slot [P:30 "first update all the black spins ... another
// kernel ... white spins"; proposal rule from BASELINE.json configs: theta' uniform in [0,2pi)].
void metropolis_pass_slot(Ctx& c, int r, int colour) {
    const int L = c.L;
    float* th = c.theta.data() + (int64_t)r * c.N;
    const uint32_t key[2] = { (uint32_t)(c.seed & 0xffffffffu), (uint32_t)(c.seed >> 32) };
    const double beta32 = (double)(float)c.beta_of_slot[r];          // reading R13
    uint64_t acc = 0;
    for (int z = 0; z < L; ++z)
      for (int y = 0; y < L; ++y)
        for (int x = 0; x < L; ++x) {
            if (((x + y + z) & 1) != colour) continue;               // reading R3: black = even
            const int64_t i = x + (int64_t)L * (y + (int64_t)L * z);
            const uint32_t ctr[4] = { (uint32_t)(i >> 2), (uint32_t)r, c.n_met,
                                      colour == 0 ? STREAM_MET_BLACK : STREAM_MET_WHITE };
            uint32_t W[4];
            philox4x32_10(ctr, key, W);
            const int p = (int)((i >> 1) & 1);                       // which of the quad's two same-colour sites
            const float theta_new = TWO_PI_F * u24(W[2 * p]);        // ONE fp32 multiply
            const float u = u24(W[2 * p + 1]);
            double hx, hy;
            local_field(c, th, x, y, z, hx, hy);
            const double t_old = (double)th[i], t_new = (double)theta_new;
            const double dE = -(hx * (std::cos(t_new) - std::cos(t_old)) +
                                hy * (std::sin(t_new) - std::sin(t_old)));   // Eq. 1
            const double prob = std::exp(-beta32 * dE);
            if (c.tr_met_p) c.tr_met_p[(int64_t)r * c.N + i] = prob;
            if (c.tr_met_u) c.tr_met_u[(int64_t)r * c.N + i] = u;
            if ((double)u < prob) { th[i] = theta_new; ++acc; }
        }
    c.met_acc[r] += acc;
}

// One over-relaxation colour pass over one slot: reflect S_i about its local field
// [P:38-43 Eq. 2], in angle form theta' = 2 phi - theta, phi = arg(h) (north_star).
void overrelax_pass_slot(Ctx& c, int r, int colour) {
    const int L = c.L;
    float* th = c.theta.data() + (int64_t)r * c.N;
    for (int z = 0; z < L; ++z)
      for (int y = 0; y < L; ++y)
        for (int x = 0; x < L; ++x) {
            if (((x + y + z) & 1) != colour) continue;
            const int64_t i = x + (int64_t)L * (y + (int64_t)L * z);
            double hx, hy;
            local_field(c, th, x, y, z, hx, hy);
            if (c.tr_or_h) c.tr_or_h[(int64_t)r * c.N + i] = std::sqrt(hx * hx + hy * hy);
            if (hx == 0.0 && hy == 0.0) continue;                    // reading R6
            double t = 2.0 * std::atan2(hy, hx) - (double)th[i];
            t = std::fmod(t, TWO_PI_D);
            if (t < 0.0) t += TWO_PI_D;                              // reading R7: [0, 2pi)
            th[i] = (float)t;                                        // rounded once to fp32
        }
}

// Observables of one slot [P:52-56 Eqs. 4-5; E_n of Eq. 3 P:47-50].
void measure_slot(const Ctx& c, int r, double out[5]) {
    const int L = c.L;
    const float* th = c.theta.data() + (int64_t)r * c.N;
    double E = 0.0, Mx = 0.0, My = 0.0;
    for (int z = 0; z < L; ++z)
      for (int y = 0; y < L; ++y)
        for (int x = 0; x < L; ++x) {
            const double t = (double)th[x + (int64_t)L * (y + (int64_t)L * z)];
            const double tx = (double)th[wrap(x + 1, L) + (int64_t)L * (y + (int64_t)L * z)];
            const double ty = (double)th[x + (int64_t)L * (wrap(y + 1, L) + (int64_t)L * z)];
            const double tz = (double)th[x + (int64_t)L * (y + (int64_t)L * wrap(z + 1, L))];
            E -= std::cos(t - tx) + std::cos(t - ty) + std::cos(t - tz);   // Eq. 1, J = 1
            Mx += std::cos(t);                                             // Eq. 4
            My += std::sin(t);
        }
    const double M2 = Mx * Mx + My * My;
    out[0] = E; out[1] = Mx; out[2] = My; out[3] = M2; out[4] = M2 * M2;   // Eq. 5 ingredients
}

// The six sums of one slot that the spin-stiffness estimator is made of [P:58-60 Eq. 6]: for each
// lattice direction mu = x, y, z, over the N bonds (i, i+mu):
//   C_mu = sum cos(theta_i - theta_{i+mu}),   S_mu = sum sin(theta_i - theta_{i+mu}).
// Eq. 6 is then rho_s = 1/(3N) sum_mu [ <C_mu> - (1/T) <S_mu^2> ] (host arithmetic on the time series).
void stiffness_slot(const Ctx& c, int r, double out[6]) {
    const int L = c.L;
    const float* th = c.theta.data() + (int64_t)r * c.N;
    double C[3] = { 0.0, 0.0, 0.0 }, S[3] = { 0.0, 0.0, 0.0 };
    for (int z = 0; z < L; ++z)
      for (int y = 0; y < L; ++y)
        for (int x = 0; x < L; ++x) {
            const double t = (double)th[x + (int64_t)L * (y + (int64_t)L * z)];
            const double tn[3] = { (double)th[wrap(x + 1, L) + (int64_t)L * (y + (int64_t)L * z)],
                                   (double)th[x + (int64_t)L * (wrap(y + 1, L) + (int64_t)L * z)],
                                   (double)th[x + (int64_t)L * (y + (int64_t)L * wrap(z + 1, L))] };
            for (int mu = 0; mu < 3; ++mu) { C[mu] += std::cos(t - tn[mu]); S[mu] += std::sin(t - tn[mu]); }
        }
    for (int mu = 0; mu < 3; ++mu) { out[mu] = C[mu]; out[3 + mu] = S[mu]; }
}

template <class F>
void for_active_slots(Ctx& c, F f) {
    const int n = (int)c.active.size();
    const int nt = c.n_threads < 1 ? 1 : (c.n_threads > n ? n : c.n_threads);
    if (nt <= 1) { for (int a = 0; a < n; ++a) f(c.active[a]); return; }
    std::vector<std::thread> pool;
    for (int t = 0; t < nt; ++t)
        pool.emplace_back([&, t]() { for (int a = t; a < n; a += nt) f(c.active[a]); });
    for (auto& th : pool) th.join();
}

}  // namespace

extern "C" {

struct xyo_ctx { Ctx c; };

void xyo_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }

xyo_ctx* xyo_create(int L, int R, const double* betas, uint64_t seed) {
    if (L < 2 || (L & 1) || R < 1 || !betas) return nullptr;
    for (int k = 0; k < R; ++k) if (!std::isfinite(betas[k])) return nullptr;
    xyo_ctx* h = new xyo_ctx;
    Ctx& c = h->c;
    c.L = L; c.R = R; c.N = (int64_t)L * L * L; c.seed = seed;
    c.betas.assign(betas, betas + R);
    c.beta_of_slot.assign(betas, betas + R);
    c.slot_at_rank.resize(R);
    c.active.resize(R);
    for (int k = 0; k < R; ++k) { c.slot_at_rank[k] = k; c.active[k] = k; }
    c.theta.assign((size_t)R * c.N, 0.0f);
    c.met_acc.assign(R, 0);
    c.pt_acc.assign(R > 1 ? R - 1 : 0, 0);
    return h;
}

void xyo_destroy(xyo_ctx* h) { delete h; }

int xyo_set_threads(xyo_ctx* h, int n) { if (!h || n < 1) return -1; h->c.n_threads = n; return 0; }

// Restrict sweeps / measure to a subset of slots (n = 0 restores all).  Used to sample the
// big configurations: replicas are independent within a sweep and the RNG is keyed by slot.
int xyo_set_active_slots(xyo_ctx* h, const int* slots, int n) {
    if (!h || n < 0 || n > h->c.R) return -1;
    Ctx& c = h->c;
    if (n == 0) { c.active.resize(c.R); for (int k = 0; k < c.R; ++k) c.active[k] = k; return 0; }
    for (int a = 0; a < n; ++a) if (slots[a] < 0 || slots[a] >= c.R) return -1;
    c.active.assign(slots, slots + n);
    return 0;
}

// Random start: theta uniform on [0, 2pi) from the INIT stream [configs: "random-start angles from seed"].
int xyo_init_random(xyo_ctx* h) {
    if (!h) return -1;
    Ctx& c = h->c;
    const uint32_t key[2] = { (uint32_t)(c.seed & 0xffffffffu), (uint32_t)(c.seed >> 32) };
    for (int r = 0; r < c.R; ++r)
        for (int64_t i = 0; i < c.N; ++i) {
            const uint32_t ctr[4] = { (uint32_t)(i >> 2), (uint32_t)r, 0u, STREAM_INIT };
            uint32_t W[4];
            philox4x32_10(ctr, key, W);
            c.theta[(size_t)r * c.N + i] = TWO_PI_F * u24(W[i & 3]);
        }
    return 0;
}

int xyo_init_ordered(xyo_ctx* h, float theta0) {                      // config 4: "ordered start (all theta=0)"
    if (!h) return -1;
    for (auto& t : h->c.theta) t = theta0;
    return 0;
}

float* xyo_state_ptr(xyo_ctx* h) { return h ? h->c.theta.data() : nullptr; }
int xyo_set_state(xyo_ctx* h, const float* s) { if (!h || !s) return -1; std::memcpy(h->c.theta.data(), s, h->c.theta.size() * sizeof(float)); return 0; }
int xyo_get_state(xyo_ctx* h, float* s) { if (!h || !s) return -1; std::memcpy(s, h->c.theta.data(), h->c.theta.size() * sizeof(float)); return 0; }

int xyo_get_perm(xyo_ctx* h, int* p) { if (!h || !p) return -1; for (int k = 0; k < h->c.R; ++k) p[k] = h->c.slot_at_rank[k]; return 0; }
int xyo_set_perm(xyo_ctx* h, const int* p) {
    if (!h || !p) return -1;
    Ctx& c = h->c;
    std::vector<int> seen(c.R, 0);
    for (int k = 0; k < c.R; ++k) { if (p[k] < 0 || p[k] >= c.R || seen[p[k]]++) return -1; }
    for (int k = 0; k < c.R; ++k) { c.slot_at_rank[k] = p[k]; c.beta_of_slot[p[k]] = c.betas[k]; }
    return 0;
}
int xyo_get_beta_of_slot(xyo_ctx* h, double* b) { if (!h || !b) return -1; for (int r = 0; r < h->c.R; ++r) b[r] = h->c.beta_of_slot[r]; return 0; }
int xyo_get_counters(xyo_ctx* h, uint32_t* n) { if (!h || !n) return -1; n[0] = h->c.n_met; n[1] = h->c.n_or; n[2] = h->c.n_pt; return 0; }
int xyo_set_counters(xyo_ctx* h, const uint32_t* n) { if (!h || !n) return -1; h->c.n_met = n[0]; h->c.n_or = n[1]; h->c.n_pt = n[2]; return 0; }
int xyo_get_accept_counts(xyo_ctx* h, uint64_t* met, uint64_t* pt) {
    if (!h) return -1;
    if (met) for (int r = 0; r < h->c.R; ++r) met[r] = h->c.met_acc[r];
    if (pt) for (int k = 0; k + 1 < h->c.R; ++k) pt[k] = h->c.pt_acc[k];
    return 0;
}
int xyo_set_trace(xyo_ctx* h, double* met_p, float* met_u, double* or_h, double* pt_p, double* pt_u) {
    if (!h) return -1;
    h->c.tr_met_p = met_p; h->c.tr_met_u = met_u; h->c.tr_or_h = or_h; h->c.tr_pt_p = pt_p; h->c.tr_pt_u = pt_u;
    return 0;
}

// A single colour pass (does not advance n_met); the sweep below is pass(0), pass(1), ++n_met.
int xyo_metropolis_pass(xyo_ctx* h, int colour) {
    if (!h || (colour != 0 && colour != 1)) return -1;
    Ctx& c = h->c;
    for_active_slots(c, [&](int r) { metropolis_pass_slot(c, r, colour); });
    return 0;
}
int xyo_metropolis_sweep(xyo_ctx* h) {                                 // black, then white
    if (!h) return -1;
    xyo_metropolis_pass(h, 0);
    xyo_metropolis_pass(h, 1);
    ++h->c.n_met;
    return 0;
}
int xyo_overrelax_pass(xyo_ctx* h, int colour) {
    if (!h || (colour != 0 && colour != 1)) return -1;
    Ctx& c = h->c;
    for_active_slots(c, [&](int r) { overrelax_pass_slot(c, r, colour); });
    return 0;
}
int xyo_overrelax_sweep(xyo_ctx* h) {                                  // reading R4: black, then white
    if (!h) return -1;
    xyo_overrelax_pass(h, 0);
    xyo_overrelax_pass(h, 1);
    ++h->c.n_or;
    return 0;
}

// out_by_slot[R][5] = E, Mx, My, |M|^2, |M|^4 of each ACTIVE slot (others left untouched).
int xyo_measure_slots(xyo_ctx* h, double* out_by_slot) {
    if (!h || !out_by_slot) return -1;
    Ctx& c = h->c;
    for_active_slots(c, [&](int r) { measure_slot(c, r, out_by_slot + 5 * (size_t)r); });
    return 0;
}
// out[R][5] indexed by RANK k (temperature), as the physics consumes it [P:62].
int xyo_measure(xyo_ctx* h, double* out) {
    if (!h || !out) return -1;
    Ctx& c = h->c;
    std::vector<double> by_slot(5 * (size_t)c.R, std::nan(""));
    xyo_measure_slots(h, by_slot.data());
    for (int k = 0; k < c.R; ++k) std::memcpy(out + 5 * (size_t)k, by_slot.data() + 5 * (size_t)c.slot_at_rank[k], 5 * sizeof(double));
    return 0;
}

// out[R][6] = Cx, Cy, Cz, Sx, Sy, Sz (see stiffness_slot) indexed by RANK k.
int xyo_measure_stiffness(xyo_ctx* h, double* out) {
    if (!h || !out) return -1;
    Ctx& c = h->c;
    std::vector<double> by_slot(6 * (size_t)c.R, std::nan(""));
    for_active_slots(c, [&](int r) { stiffness_slot(c, r, by_slot.data() + 6 * (size_t)r); });
    for (int k = 0; k < c.R; ++k) std::memcpy(out + 6 * (size_t)k, by_slot.data() + 6 * (size_t)c.slot_at_rank[k], 6 * sizeof(double));
    return 0;
}

// Replica exchange with the energies given per slot [P:45-50 Eq. 3]; pairs (k,k+1) with
// k = n_pt mod 2, +2, ... (reading R9); beta labels are swapped, never spin arrays (R11).
int xyo_pt_exchange_with_E(xyo_ctx* h, const double* E_by_slot) {
    if (!h || !E_by_slot) return -1;
    Ctx& c = h->c;
    const uint32_t key[2] = { (uint32_t)(c.seed & 0xffffffffu), (uint32_t)(c.seed >> 32) };
    if (c.tr_pt_p) for (int k = 0; k + 1 < c.R; ++k) c.tr_pt_p[k] = std::nan("");
    if (c.tr_pt_u) for (int k = 0; k + 1 < c.R; ++k) c.tr_pt_u[k] = std::nan("");
    for (int k = (int)(c.n_pt & 1u); k + 1 < c.R; k += 2) {
        const int a = c.slot_at_rank[k], b = c.slot_at_rank[k + 1];
        const uint32_t ctr[4] = { (uint32_t)k, 0u, c.n_pt, STREAM_PT };
        uint32_t W[4];
        philox4x32_10(ctr, key, W);
        const double u = (double)W[0] * (1.0 / 4294967296.0);
        const double prob = std::exp((c.betas[k] - c.betas[k + 1]) * (E_by_slot[a] - E_by_slot[b]));   // Eq. 3
        if (c.tr_pt_p) c.tr_pt_p[k] = prob;
        if (c.tr_pt_u) c.tr_pt_u[k] = u;
        if (u < prob) {
            c.slot_at_rank[k] = b; c.slot_at_rank[k + 1] = a;
            c.beta_of_slot[a] = c.betas[k + 1]; c.beta_of_slot[b] = c.betas[k];
            ++c.pt_acc[k];
        }
    }
    ++c.n_pt;
    return 0;
}
int xyo_pt_exchange(xyo_ctx* h) {
    if (!h) return -1;
    Ctx& c = h->c;
    std::vector<double> by_slot(5 * (size_t)c.R, 0.0);
    std::vector<int> saved = c.active;                         // E of every slot is needed
    xyo_set_active_slots(h, nullptr, 0);
    xyo_measure_slots(h, by_slot.data());
    c.active = saved;
    std::vector<double> E(c.R);
    for (int r = 0; r < c.R; ++r) E[r] = by_slot[5 * (size_t)r];
    return xyo_pt_exchange_with_E(h, E.data());
}

}  // extern "C"
