// xy_kernels.cuh -- the sm_100a kernels of the XY Monte Carlo step.
//
// Data layout in HBM: colour-split, replica-major fp32 angles
//     theta_c[slot][z][y][xh],  c = (x+y+z)&1,  xh = x>>1,  row length W = L/2 floats
// so a colour pass reads both half-lattices once and writes only its own: 12 B per site-update.
//
// One kernel skeleton serves Metropolis (a2), over-relaxation (a3) and the observable reduction
// (a4).  A thread block owns a tile of TY full rows of its colour and MARCHES through TZ planes.
// Per plane it (1) turns the other colour's TY+2 rows of the next plane into (cos, sin) ONCE and
// parks them in a 4-deep ring of shared-memory planes, (2) __syncthreads, (3) updates its own
// plane from the three staged planes z-1, z, z+1.  Each thread owns four consecutive sites
// (one 128-bit load and store) of one row for the whole march; x wraps inside the tile, y and z
// wrap in the global addresses of the staged rows.  The next plane's global loads are issued
// before the current plane is computed.
#pragma once
#include "xy_device.cuh"

namespace xyk {

enum { MODE_MET = 0, MODE_OR = 1, MODE_MEASURE = 2 };

struct SweepParams {
    float* own;                  // colour array being updated   [R][L][L][W]
    const float* other;          // the other colour's array (read only during the pass)
    int L, W, W4;                // W = L/2 floats per row, W4 = L/8 float4 per row
    int TY, TZ, nTY, nTZ;        // tile rows, march length, tiles per replica in y and z
    int colour;                  // colour of `own`
    int nItems;                  // TY * W4 own float4 per plane (<= blockDim.x)
    size_t half_n;               // L^3 / 2 floats per slot per colour
    PhiloxKeys keys;
    uint32_t sweep;              // n_met (Philox counter word 2)
    const float* beta32_of_slot; // Metropolis: fp32 beta label per slot (R13)
    unsigned long long* met_acc; // Metropolis: accepted proposals per slot
    unsigned long long* exact_count;  // Metropolis: decisions re-evaluated in fp64
    float* trace;                // Metropolis test hook: p_fast per own site (same layout as own) or null
    double* partials;            // measure: [R][nTY*nTZ][3] partial E, Mx, My
};

__device__ __forceinline__ float4 ldg4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }

template <int MODE, bool TRACE>
__global__ void __launch_bounds__(512) sweep_kernel(const SweepParams P) {
    extern __shared__ __align__(16) float smem[];
    const int L = P.L, W = P.W, W4 = P.W4, TY = P.TY, TZ = P.TZ;
    const int planeS = (TY + 2) * W;                 // floats per staged plane (per component)
    float* const sC = smem;                          // cos ring: 4 planes
    float* const sS = smem + 4 * planeS;             // sin ring: 4 planes

    const int tid = threadIdx.x;
    const int slot = blockIdx.y;
    const int tile = blockIdx.x;
    const int tzi = tile / P.nTY, tyi = tile - tzi * P.nTY;
    const int y0 = tyi * TY, z0 = tzi * TZ;

    const float* __restrict__ other = P.other + (size_t)slot * P.half_n;
    float* __restrict__ own = P.own + (size_t)slot * P.half_n;

    // this thread's own item: row ty of the tile, float4 column q
    const bool active = tid < P.nItems;
    const int ty = active ? tid / W4 : 0;
    const int q = active ? tid - ty * W4 : 0;
    const int col = 4 * q;
    const int y = y0 + ty;

    // staging duty 1: staged row ty (global y0-1+ty), column q.  Duty 2 (tid < 2*W4): staged rows TY, TY+1.
    int ys1 = y - 1; if (ys1 < 0) ys1 += L;
    const bool duty2 = tid < 2 * W4;
    const int r2 = duty2 ? tid / W4 : 0;             // 0 or 1
    const int q2 = duty2 ? tid - r2 * W4 : 0;
    int ys2 = y0 + TY - 1 + r2; if (ys2 >= L) ys2 -= L;
    const int sOff1 = ty * W + col;                  // float offset inside a staged plane
    const int sOff2 = (TY + r2) * W + 4 * q2;
    const size_t gRow1 = (size_t)ys1 * W + col;      // + z*L*W
    const size_t gRow2 = (size_t)ys2 * W + 4 * q2;
    const size_t gOwn = (size_t)y * W + col;
    const size_t planeG = (size_t)L * W;

    // measure: which staged items are "mine" (non-halo) for the magnetisation of the other colour
    const bool m1_rowok = active && ty >= 1;         // staged row ty in [1, TY]
    const bool m2_rowok = duty2 && r2 == 0;          // staged row TY
    float accE = 0.f, accMx = 0.f, accMy = 0.f;      // per-plane fp32, flushed to double each plane
    double dE = 0.0, dMx = 0.0, dMy = 0.0;

    auto plane_of = [&](int j) { int z = z0 - 1 + j; if (z < 0) z += L; if (z >= L) z -= L; return z; };
    auto stage = [&](const float4& v, int j, int sOff, bool count_m) {
        float4 c, s;
        fast_sincos(v.x, s.x, c.x); fast_sincos(v.y, s.y, c.y);
        fast_sincos(v.z, s.z, c.z); fast_sincos(v.w, s.w, c.w);
        const int base = (j & 3) * planeS + sOff;
        *reinterpret_cast<float4*>(sC + base) = c;
        *reinterpret_cast<float4*>(sS + base) = s;
        if (MODE == MODE_MEASURE && count_m) {
            accMx += (c.x + c.y) + (c.z + c.w);
            accMy += (s.x + s.y) + (s.z + s.w);
        }
    };

    // ---- prologue: planes j = 0, 1 staged; j = 2 and own plane 0 in flight -----------------
    float4 o1 = make_float4(0, 0, 0, 0), o2 = o1, mine = o1;
#pragma unroll
    for (int j = 0; j < 2; ++j) {
        const size_t zb = (size_t)plane_of(j) * planeG;
        if (active) { o1 = ldg4(other + zb + gRow1); }
        if (duty2) { o2 = ldg4(other + zb + gRow2); }
        if (active) stage(o1, j, sOff1, m1_rowok && j >= 1);
        if (duty2) stage(o2, j, sOff2, m2_rowok && j >= 1);
    }
    {
        const size_t zb = (size_t)plane_of(2) * planeG;
        if (active) { o1 = ldg4(other + zb + gRow1); mine = *reinterpret_cast<const float4*>(own + (size_t)z0 * planeG + gOwn); }
        if (duty2) { o2 = ldg4(other + zb + gRow2); }
    }

    float bl = 0.f, window = 0.f, beta32 = 0.f;
    if (MODE == MODE_MET) {
        beta32 = P.beta32_of_slot[slot];
        bl = beta32 * 1.44269504f;                   // exp(beta g) = 2^(bl g)
        window = fabsf(beta32) * 1.4e-4f + 1e-6f;    // see kExactWindow in xy_device.cuh
    }
    unsigned int nacc = 0, nexact = 0;
    const uint32_t quad_row = (uint32_t)(L >> 2);
    const uint32_t stream = P.colour == 0 ? kStreamMetBlack : kStreamMetWhite;

    // ---- march ---------------------------------------------------------------------------
    for (int zi = 0; zi < TZ; ++zi) {
        const int z = z0 + zi;
        if (active) stage(o1, zi + 2, sOff1, m1_rowok && zi + 2 <= TZ);
        if (duty2) stage(o2, zi + 2, sOff2, m2_rowok && zi + 2 <= TZ);
        const float4 cur = mine;
        if (zi + 1 < TZ) {                           // prefetch for the next plane
            const size_t zb = (size_t)plane_of(zi + 3) * planeG;
            if (active) { o1 = ldg4(other + zb + gRow1); mine = *reinterpret_cast<const float4*>(own + (size_t)(z + 1) * planeG + gOwn); }
            if (duty2) { o2 = ldg4(other + zb + gRow2); }
        }
        __syncthreads();
        if (active) {
            const float* cM = sC + ((zi) & 3) * planeS;       // plane z-1
            const float* cZ = sC + ((zi + 1) & 3) * planeS;   // plane z
            const float* cP = sC + ((zi + 2) & 3) * planeS;   // plane z+1
            const float* sM = sS + ((zi) & 3) * planeS;
            const float* sZ = sS + ((zi + 1) & 3) * planeS;
            const float* sP = sS + ((zi + 2) & 3) * planeS;
            const int rC = (ty + 1) * W + col, rM = ty * W + col, rP = (ty + 2) * W + col;
            const int par = (y + z + P.colour) & 1;           // x parity of this row's own sites
            const int ecol = par ? (col + 4 == W ? 0 : col + 4) : (col == 0 ? W - 1 : col - 1);
            float hx[4], hy[4];
            {
                const float4 c = *reinterpret_cast<const float4*>(cZ + rC);
                const float e = cZ[(ty + 1) * W + ecol];
                const float4 a = *reinterpret_cast<const float4*>(cZ + rM);
                const float4 b = *reinterpret_cast<const float4*>(cZ + rP);
                const float4 d = *reinterpret_cast<const float4*>(cM + rC);
                const float4 f = *reinterpret_cast<const float4*>(cP + rC);
                const float s01 = c.x + c.y, s12 = c.y + c.z, s23 = c.z + c.w;
                const float se = e + (par ? c.w : c.x);
                hx[0] = (par ? s01 : se) + (a.x + b.x) + (d.x + f.x);
                hx[1] = (par ? s12 : s01) + (a.y + b.y) + (d.y + f.y);
                hx[2] = (par ? s23 : s12) + (a.z + b.z) + (d.z + f.z);
                hx[3] = (par ? se : s23) + (a.w + b.w) + (d.w + f.w);
            }
            {
                const float4 c = *reinterpret_cast<const float4*>(sZ + rC);
                const float e = sZ[(ty + 1) * W + ecol];
                const float4 a = *reinterpret_cast<const float4*>(sZ + rM);
                const float4 b = *reinterpret_cast<const float4*>(sZ + rP);
                const float4 d = *reinterpret_cast<const float4*>(sM + rC);
                const float4 f = *reinterpret_cast<const float4*>(sP + rC);
                const float s01 = c.x + c.y, s12 = c.y + c.z, s23 = c.z + c.w;
                const float se = e + (par ? c.w : c.x);
                hy[0] = (par ? s01 : se) + (a.x + b.x) + (d.x + f.x);
                hy[1] = (par ? s12 : s01) + (a.y + b.y) + (d.y + f.y);
                hy[2] = (par ? s23 : s12) + (a.z + b.z) + (d.z + f.z);
                hy[3] = (par ? se : s23) + (a.w + b.w) + (d.w + f.w);
            }
            float th[4] = { cur.x, cur.y, cur.z, cur.w };

            if (MODE == MODE_MET) {
                const uint32_t c0 = (uint32_t)(col >> 1) + quad_row * (uint32_t)(y + L * z);
                uint32_t w[8];
                {
                    uint32_t t4[4];
                    philox4x32_10(c0, (uint32_t)slot, P.sweep, stream, P.keys, t4);
                    w[0] = t4[0]; w[1] = t4[1]; w[2] = t4[2]; w[3] = t4[3];
                    philox4x32_10(c0 + 1, (uint32_t)slot, P.sweep, stream, P.keys, t4);
                    w[4] = t4[0]; w[5] = t4[1]; w[6] = t4[2]; w[7] = t4[3];
                }
                float ptrace[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const float tn = word_to_angle(w[2 * k]);
                    const float u = word_to_u24(w[2 * k + 1]);
                    float so, co, sn, cn;
                    fast_sincos(th[k], so, co);
                    fast_sincos(tn, sn, cn);
                    const float g = fmaf(hx[k], cn - co, hy[k] * (sn - so));   // = -dE
                    const float pf = fast_ex2(bl * g);
                    bool acc = u < pf;
                    if (fabsf(u - pf) < window) {
                        acc = metropolis_exact(other, L, W, par, col + k, y, z, th[k], tn, u, beta32);
                        ++nexact;
                    }
                    if (TRACE) ptrace[k] = fminf(pf, 3.0e38f);
                    if (acc) { th[k] = tn; ++nacc; }
                }
                if (TRACE) {
                    float* tr = P.trace + (size_t)P.colour * gridDim.y * P.half_n + (size_t)slot * P.half_n;
                    *reinterpret_cast<float4*>(tr + (size_t)z * planeG + gOwn) = make_float4(ptrace[0], ptrace[1], ptrace[2], ptrace[3]);
                }
                *reinterpret_cast<float4*>(own + (size_t)z * planeG + gOwn) = make_float4(th[0], th[1], th[2], th[3]);
            } else if (MODE == MODE_OR) {
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    if (hx[k] != 0.0f || hy[k] != 0.0f) {                      // R6
                        float t = fmaf(2.0f, fast_atan2_pos(hy[k], hx[k]), -th[k]);
                        t = (t < 0.0f) ? t + kTwoPiF : t;
                        t = (t >= kTwoPiF) ? t - kTwoPiF : t;
                        th[k] = t;
                    }
                }
                *reinterpret_cast<float4*>(own + (size_t)z * planeG + gOwn) = make_float4(th[0], th[1], th[2], th[3]);
            } else {  // MODE_MEASURE: own = white; E = -sum_white S_i . h_i counts every bond once
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    float s, c;
                    fast_sincos(th[k], s, c);
                    accE = fmaf(c, hx[k], fmaf(s, hy[k], accE));
                    accMx += c; accMy += s;
                }
            }
        }
        if (MODE == MODE_MEASURE) {
            dE += (double)accE; dMx += (double)accMx; dMy += (double)accMy;
            accE = accMx = accMy = 0.f;
        }
    }

    // ---- epilogue ---------------------------------------------------------------------------
    if (MODE == MODE_MET) {
        unsigned int a = nacc, e = nexact;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, o); e += __shfl_xor_sync(0xffffffffu, e, o); }
        if ((tid & 31) == 0) {
            if (a) atomicAdd(P.met_acc + slot, (unsigned long long)a);
            if (e) atomicAdd(P.exact_count, (unsigned long long)e);
        }
    }
    if (MODE == MODE_MEASURE) {
        // fixed-order block reduction in double: warp shuffle tree, then warp 0 sums the warps in order
        __shared__ double red[3][32];
        double v[3] = { dE, dMx, dMy };
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v[c] += __shfl_xor_sync(0xffffffffu, v[c], o);
        __syncthreads();
        const int wid = tid >> 5, nw = (blockDim.x + 31) >> 5;
        if ((tid & 31) == 0) { red[0][wid] = v[0]; red[1][wid] = v[1]; red[2][wid] = v[2]; }
        __syncthreads();
        if (tid < 3) {
            double s = 0.0;
            for (int k = 0; k < nw; ++k) s += red[tid][k];
            P.partials[((size_t)slot * gridDim.x + tile) * 3 + tid] = tid == 0 ? -s : s;
        }
    }
}

// Final stage of a4: block k sums the tile partials of slot_at_rank[k] in fixed order and writes
// the five observables by rank and by slot.
__global__ void measure_finalize_kernel(const double* __restrict__ partials, int n_tiles,
                                        const int* __restrict__ slot_at_rank,
                                        double* __restrict__ obs_rank, double* __restrict__ obs_slot,
                                        double* __restrict__ series_row) {
    const int k = blockIdx.x;
    const int slot = slot_at_rank[k];
    __shared__ double red[3][32];
    double v[3] = { 0.0, 0.0, 0.0 };
    for (int t = threadIdx.x; t < n_tiles; t += blockDim.x)
        for (int c = 0; c < 3; ++c) v[c] += partials[((size_t)slot * n_tiles + t) * 3 + c];
    for (int c = 0; c < 3; ++c)
        for (int o = 16; o > 0; o >>= 1) v[c] += __shfl_xor_sync(0xffffffffu, v[c], o);
    const int wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    if ((threadIdx.x & 31) == 0) for (int c = 0; c < 3; ++c) red[c][wid] = v[c];
    __syncthreads();
    if (threadIdx.x == 0) {
        double s[3] = { 0.0, 0.0, 0.0 };
        for (int w = 0; w < nw; ++w) for (int c = 0; c < 3; ++c) s[c] += red[c][w];
        const double m2 = s[1] * s[1] + s[2] * s[2];
        const double o5[5] = { s[0], s[1], s[2], m2, m2 * m2 };
        for (int c = 0; c < 5; ++c) {
            obs_rank[5 * k + c] = o5[c];
            obs_slot[5 * slot + c] = o5[c];
            if (series_row) series_row[5 * k + c] = o5[c];
        }
    }
}

// a5: one replica exchange (Eq. 3) in fp64; thread per candidate pair.
__global__ void pt_exchange_kernel(int R, uint32_t n_pt, PhiloxKeys keys, const double* __restrict__ betas,
                                   const double* __restrict__ obs_slot, int* __restrict__ slot_at_rank,
                                   double* __restrict__ beta_of_slot, float* __restrict__ beta32_of_slot,
                                   unsigned long long* __restrict__ pt_acc) {
    const int pair = blockIdx.x * blockDim.x + threadIdx.x;
    const int k = (int)(n_pt & 1u) + 2 * pair;
    if (k + 1 >= R) return;
    const int a = slot_at_rank[k], b = slot_at_rank[k + 1];
    uint32_t w[4];
    philox4x32_10((uint32_t)k, 0u, n_pt, kStreamPT, keys, w);
    const double u = (double)w[0] * (1.0 / 4294967296.0);
    const double prob = exp((betas[k] - betas[k + 1]) * (obs_slot[5 * a] - obs_slot[5 * b]));
    if (u < prob) {
        slot_at_rank[k] = b; slot_at_rank[k + 1] = a;
        beta_of_slot[a] = betas[k + 1]; beta_of_slot[b] = betas[k];
        beta32_of_slot[a] = (float)betas[k + 1]; beta32_of_slot[b] = (float)betas[k];
        pt_acc[k] += 1ull;
    }
}

// a0: random start from the INIT stream; one thread per natural quad of four consecutive x.
__global__ void init_random_kernel(float* __restrict__ black, float* __restrict__ white, int L, int R,
                                   PhiloxKeys keys) {
    const size_t n_quads = (size_t)R * L * L * (L >> 2);
    const int W = L >> 1;
    for (size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x; g < n_quads; g += (size_t)gridDim.x * blockDim.x) {
        const int xq = (int)(g % (size_t)(L >> 2));
        size_t rest = g / (size_t)(L >> 2);
        const int y = (int)(rest % L); rest /= L;
        const int z = (int)(rest % L);
        const int r = (int)(rest / L);
        const uint32_t c0 = (uint32_t)xq + (uint32_t)(L >> 2) * (uint32_t)(y + L * z);
        uint32_t w[4];
        philox4x32_10(c0, (uint32_t)r, 0u, kStreamInit, keys, w);
        const float t0 = word_to_angle(w[0]), t1 = word_to_angle(w[1]), t2 = word_to_angle(w[2]), t3 = word_to_angle(w[3]);
        // x = 4xq+j has colour (j+y+z)&1 and xh = 2xq + (j>>1)
        const int par = (y + z) & 1;                 // colour of x = 4xq
        const size_t o = (((size_t)r * L + z) * L + y) * W + 2 * xq;
        const float2 evens = make_float2(t0, t2), odds = make_float2(t1, t3);
        *reinterpret_cast<float2*>((par == 0 ? black : white) + o) = evens;
        *reinterpret_cast<float2*>((par == 0 ? white : black) + o) = odds;
    }
}

__global__ void fill_kernel(float* __restrict__ p, size_t n, float v) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) p[i] = v;
}

// natural [slots][z][y][x] <-> colour-split; one thread per 8 consecutive x (two float4 natural,
// one float4 per colour).  `slot0` offsets the split arrays (natural points at slot0's first site).
template <bool TO_SPLIT>
__global__ void convert_kernel(float* __restrict__ natural, float* __restrict__ black, float* __restrict__ white,
                               int L, int n_slots, int slot0) {
    const int W4 = L >> 3;
    const size_t n_items = (size_t)n_slots * L * L * W4;
    for (size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x; g < n_items; g += (size_t)gridDim.x * blockDim.x) {
        const int q = (int)(g % (size_t)W4);
        size_t rest = g / (size_t)W4;
        const int y = (int)(rest % L); rest /= L;
        const int z = (int)(rest % L);
        const int par = (y + z) & 1;                 // colour of even x in this row
        float4* nat = reinterpret_cast<float4*>(natural) + 2 * g;
        const size_t so = (size_t)slot0 * L * L * W4 + g;         // float4 index in the split arrays
        float4* ev = reinterpret_cast<float4*>(par == 0 ? black : white) + so;   // even x
        float4* od = reinterpret_cast<float4*>(par == 0 ? white : black) + so;   // odd x
        if (TO_SPLIT) {
            const float4 a = nat[0], b = nat[1];
            *ev = make_float4(a.x, a.z, b.x, b.z);
            *od = make_float4(a.y, a.w, b.y, b.w);
        } else {
            const float4 e = *ev, o = *od;
            nat[0] = make_float4(e.x, o.x, e.y, o.y);
            nat[1] = make_float4(e.z, o.z, e.w, o.w);
        }
    }
}

// test hooks
__global__ void debug_sincos_kernel(const float* x, float* c, float* s, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        float ss, cc; fast_sincos(x[i], ss, cc); c[i] = cc; s[i] = ss;
    }
}
__global__ void debug_atan2_kernel(const float* y, const float* x, float* phi, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        phi[i] = fast_atan2_pos(y[i], x[i]);
}
__global__ void debug_philox_kernel(const uint32_t* ctr, PhiloxKeys keys, uint32_t* out, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        uint32_t w[4];
        philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], keys, w);
        out[4 * i] = w[0]; out[4 * i + 1] = w[1]; out[4 * i + 2] = w[2]; out[4 * i + 3] = w[3];
    }
}

}  // namespace xyk
