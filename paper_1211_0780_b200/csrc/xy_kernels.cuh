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
    unsigned int half_n;         // L^3 / 2 floats per slot per colour
    PhiloxKeys keys;
    uint32_t sweep;              // n_met (Philox counter word 2)
    const float* beta32_of_slot; // Metropolis: fp32 beta label per slot (R13)
    unsigned long long* met_acc; // Metropolis: accepted proposals per slot
    unsigned long long* exact_count;  // Metropolis: decisions re-evaluated in fp64
    float* trace;                // Metropolis test hook: p_fast per own site (same layout as own) or null
    double* partials;            // measure: [R][nTY*nTZ][3] partial E, Mx, My
    uint4* near_queue;           // Metropolis: decisions too close to call in fp32 (see met_fixup_kernel)
    unsigned int* near_count;    // entries appended so far in this colour pass
    unsigned int near_cap;       // capacity of near_queue
};

// Two fp32 in one 64-bit register pair: sm_100a has packed fp32 arithmetic (FADD2 / FMUL2 / FFMA2),
// one issue slot for two additions.  A staged site is the pair (cos theta, sin theta).
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) { f32x2 d; asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi)); return d; }
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }

__device__ __forceinline__ float4 ldg4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }

// Shared-memory plane: (TY+2) staged rows of the other colour, global rows y0-1 .. y0+TY.  A row of
// W = 4*W4 sites is stored as two arrays of W4 x 16 bytes: part A holds the (cos, sin) pairs of sites
// 4q, 4q+1, part B those of sites 4q+2, 4q+3, so that consecutive lanes read consecutive 16-byte
// words (no bank conflicts) and a thread's four sites are two 128-bit loads.
//
// PARMODE: 0 / 1 = the x parity of this thread's own sites is that constant on the first plane of
// the march and alternates from plane to plane (the launcher maps whole warps to rows of one
// parity class); 2 = computed per thread and plane (tiles too small for the warp-uniform mapping).
// EXACT_INLINE (Metropolis only): re-evaluate close decisions in fp64 on the spot (function call in
// the loop: slow; chosen by the launcher when |beta| is so large that most decisions are "close").
// Otherwise close decisions are appended to a global queue and settled by met_fixup_kernel, which
// keeps the fp64 code and its registers out of this loop.
template <int MODE, bool TRACE, bool FUSED, bool UNI, bool EXACT_INLINE>
__global__ void __launch_bounds__(512, 2) sweep_kernel(const SweepParams P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int L = P.L, W = P.W, W4 = P.W4, TY = P.TY, TZ = P.TZ;
    const int rowB = W * 8;                          // bytes per staged row (W pairs)
    const int planeB = (TY + 2) * rowB;              // bytes per staged plane; ring of 4 planes
    const int partB = W4 * 16;                       // byte offset of part B inside a row

    const int tid = threadIdx.x;
    const int slot = blockIdx.y;
    const int tile = blockIdx.x;
    const int tzi = tile / P.nTY, tyi = tile - tzi * P.nTY;
    const int y0 = tyi * TY, z0 = tzi * TZ;

    const float* __restrict__ other = P.other + (size_t)slot * P.half_n;
    float* __restrict__ own = P.own + (size_t)slot * P.half_n;

    // ---- this thread's own item: row ty of the tile, float4 column q ---------------------------
    const bool active = UNI || tid < P.nItems;
    int ty, q;
    if (UNI) {                                       // warps [0, n/2) take even rows, the rest odd rows
        const int half = P.nItems >> 1;
        const int cls = tid >= half;
        const int r = tid - (cls ? half : 0);
        const int t2 = r / W4;
        ty = 2 * t2 + cls; q = r - t2 * W4;
    } else {
        ty = active ? tid / W4 : 0; q = active ? tid - ty * W4 : 0;
    }
    const int col = 4 * q;
    const int y = y0 + ty;

    // staging duty 1: the other colour's float4 at this thread's own (y, q) -> staged row ty+1.
    // duty 2 (tid < 2*W4): the halo rows, staged row 0 (global y0-1) and TY+1 (global y0+TY).
    const bool duty2 = tid < 2 * W4;
    const int r2 = duty2 ? tid / W4 : 0;             // 0 or 1
    const int q2 = duty2 ? tid - r2 * W4 : 0;
    int ys2 = r2 ? y0 + TY : y0 - 1;
    if (ys2 < 0) ys2 += L;
    if (ys2 >= L) ys2 -= L;
    const int sOff1 = (ty + 1) * rowB + q * 16;      // byte offset inside a staged plane (part A)
    const int sOff2 = (r2 ? TY + 1 : 0) * rowB + q2 * 16;
    const unsigned int planeG = (unsigned int)L * W;
    const unsigned int gOwn = (unsigned int)y * W + col;       // + z*planeG: this thread's float4 in either colour array
    const unsigned int gRow2 = (unsigned int)ys2 * W + 4 * q2;

    // measure: which staged items are inside the tile (non-halo) for the other colour's magnetisation
    constexpr bool MEAS = (MODE == MODE_MEASURE) || FUSED;
    f32x2 accM = 0ull;                               // per-plane fp32 (Mx, My), flushed to double each plane
    float accE = 0.f;
    double dE = 0.0, dMx = 0.0, dMy = 0.0;

    auto plane_of = [&](int j) { int z = z0 - 1 + j; if (z < 0) z += L; if (z >= L) z -= L; return z; };
    auto stage = [&](const float4& v, int j, int sOff, bool count_m) {
        float c0, s0, c1, s1, c2, s2, c3, s3;
        fast_sincos(v.x, s0, c0); fast_sincos(v.y, s1, c1);
        fast_sincos(v.z, s2, c2); fast_sincos(v.w, s3, c3);
        const f32x2 p0 = pack2(c0, s0), p1 = pack2(c1, s1), p2 = pack2(c2, s2), p3 = pack2(c3, s3);
        unsigned char* base = smem_raw + (j & 3) * planeB + sOff;
        *reinterpret_cast<ulonglong2*>(base) = make_ulonglong2(p0, p1);
        *reinterpret_cast<ulonglong2*>(base + partB) = make_ulonglong2(p2, p3);
        if (MEAS && count_m) accM = add2(accM, add2(add2(p0, p1), add2(p2, p3)));
    };

    // ---- prologue: planes j = 0, 1 staged; j = 2 and own plane 0 in flight -----------------
    float4 o1 = make_float4(0, 0, 0, 0), o2 = o1, mine = o1;
#pragma unroll
    for (int j = 0; j < 2; ++j) {
        const unsigned int zb = (unsigned int)plane_of(j) * planeG;
        if (active) { o1 = ldg4(other + zb + gOwn); }
        if (duty2) { o2 = ldg4(other + zb + gRow2); }
        if (active) stage(o1, j, sOff1, j >= 1);
        if (duty2) stage(o2, j, sOff2, false);
    }
    {
        const unsigned int zb = (unsigned int)plane_of(2) * planeG;
        if (active) { o1 = ldg4(other + zb + gOwn); mine = *reinterpret_cast<const float4*>(own + (unsigned int)z0 * planeG + gOwn); }
        if (duty2) { o2 = ldg4(other + zb + gRow2); }
    }

    float bl = 0.f, win24 = 0.f, beta32 = 0.f;
    if (MODE == MODE_MET) {
        beta32 = P.beta32_of_slot[slot];
        bl = beta32 * 1.44269504f;                   // exp(beta g) = 2^(bl g)
        win24 = (fabsf(beta32) * kWindowPerBeta + kWindowAbs) * 16777216.0f;    // see xy_device.cuh
    }
    unsigned int nacc = 0, nexact = 0;
    const uint32_t quad_row = (uint32_t)(L >> 2);
    const uint32_t stream = P.colour == 0 ? kStreamMetBlack : kStreamMetWhite;
    // x parity of this row's own sites on plane z: (y + z + colour) & 1
    const int par0 = (y + z0 + P.colour) & 1;
    // edge pair of the row: par = 0 needs site col-1 (part B of column q-1, second pair),
    // par = 1 needs site col+4 (part A of column q+1, first pair); x wraps inside the row.
    const int eOff0 = partB + (q == 0 ? W4 - 1 : q - 1) * 16 + 8;
    const int eOff1 = (q + 1 == W4 ? 0 : q + 1) * 16;

    // ---- one plane of the march ------------------------------------------------------------------
    auto plane = [&](const int zi, const int par) {
        const int z = z0 + zi;
        if (active) stage(o1, zi + 2, sOff1, zi + 2 <= TZ);
        if (duty2) stage(o2, zi + 2, sOff2, false);
        const float4 cur = mine;
        if (zi + 1 < TZ) {                           // prefetch for the next plane
            const unsigned int zb = (unsigned int)plane_of(zi + 3) * planeG;
            if (active) { o1 = ldg4(other + zb + gOwn); mine = *reinterpret_cast<const float4*>(own + (unsigned int)(z + 1) * planeG + gOwn); }
            if (duty2) { o2 = ldg4(other + zb + gRow2); }
        }
        __syncthreads();
        if (active) {
            const unsigned char* bM = smem_raw + ((zi) & 3) * planeB;       // plane z-1
            const unsigned char* bZ = smem_raw + ((zi + 1) & 3) * planeB;   // plane z
            const unsigned char* bP = smem_raw + ((zi + 2) & 3) * planeB;   // plane z+1
            const int rC = sOff1;                                           // staged row ty+1, part A, column q
            const ulonglong2 cA = *reinterpret_cast<const ulonglong2*>(bZ + rC);
            const ulonglong2 cB = *reinterpret_cast<const ulonglong2*>(bZ + rC + partB);
            const f32x2 e = *reinterpret_cast<const f32x2*>(bZ + (ty + 1) * rowB + (par ? eOff1 : eOff0));
            const ulonglong2 aA = *reinterpret_cast<const ulonglong2*>(bZ + rC - rowB);
            const ulonglong2 aB = *reinterpret_cast<const ulonglong2*>(bZ + rC - rowB + partB);
            const ulonglong2 bA = *reinterpret_cast<const ulonglong2*>(bZ + rC + rowB);
            const ulonglong2 bB = *reinterpret_cast<const ulonglong2*>(bZ + rC + rowB + partB);
            const ulonglong2 dA = *reinterpret_cast<const ulonglong2*>(bM + rC);
            const ulonglong2 dB = *reinterpret_cast<const ulonglong2*>(bM + rC + partB);
            const ulonglong2 fA = *reinterpret_cast<const ulonglong2*>(bP + rC);
            const ulonglong2 fB = *reinterpret_cast<const ulonglong2*>(bP + rC + partB);
            // x neighbours: par = 0 -> sites (j-1, j), par = 1 -> sites (j, j+1) of the same row
            const f32x2 s01 = add2(cA.x, cA.y), s12 = add2(cA.y, cB.x), s23 = add2(cB.x, cB.y);
            const f32x2 se = add2(e, par ? cB.y : cA.x);
            f32x2 h[4];
            h[0] = add2(add2(par ? s01 : se, add2(aA.x, bA.x)), add2(dA.x, fA.x));
            h[1] = add2(add2(par ? s12 : s01, add2(aA.y, bA.y)), add2(dA.y, fA.y));
            h[2] = add2(add2(par ? s23 : s12, add2(aB.x, bB.x)), add2(dB.x, fB.x));
            h[3] = add2(add2(par ? se : s23, add2(aB.y, bB.y)), add2(dB.y, fB.y));
            float th[4] = { cur.x, cur.y, cur.z, cur.w };
            float* const gp = own + (unsigned int)z * planeG + gOwn;

            if (MODE == MODE_MET) {
                const uint32_t c0 = (uint32_t)(col >> 1) + quad_row * (uint32_t)(y + L * z);
                float ptrace[4];
#pragma unroll
                for (int pr = 0; pr < 2; ++pr) {
                    uint32_t w[4];
                    philox4x32_10(c0 + pr, (uint32_t)slot, P.sweep, stream, P.keys, w);
#pragma unroll
                    for (int kk = 0; kk < 2; ++kk) {
                        const int k = 2 * pr + kk;
                        const float kf = (float)(w[2 * kk] >> 8);
                        const float tn = kf * kTwoPiU24;
                        const float uf = (float)(w[2 * kk + 1] >> 8);            // u24 * 2^24
                        float hx, hy, so, co, sn, cn;
                        unpack2(h[k], hx, hy);
                        fast_sincos(th[k], so, co);
                        fast_sincos(tn, sn, cn);
                        const float g = fmaf(hx, cn - co, hy * (sn - so));       // = -dE
                        const float pf = fast_ex2(fmaf(bl, g, 24.0f));            // p * 2^24
                        bool acc = uf < pf;
                        if (fabsf(uf - pf) < win24) {
                            if (EXACT_INLINE) {
                                acc = metropolis_exact(other, L, W, par, col + k, y, z, th[k], tn, uf * kInvU24, beta32);
                                ++nexact;
                            } else {
                                const unsigned int e = atomicAdd(P.near_count, 1u);
                                if (e < P.near_cap)
                                    P.near_queue[e] = make_uint4(((unsigned int)z * planeG + gOwn + k) | (acc ? 0x80000000u : 0u),
                                                                 (unsigned int)slot, __float_as_uint(th[k]), 0u);
                            }
                        }
                        if (TRACE) ptrace[k] = fminf(pf * kInvU24, 3.0e38f);
                        if (acc) { th[k] = tn; ++nacc; }
                    }
                }
                if (TRACE) {
                    float* tr = P.trace + (size_t)P.colour * gridDim.y * P.half_n + (size_t)slot * P.half_n;
                    *reinterpret_cast<float4*>(tr + (unsigned int)z * planeG + gOwn) = make_float4(ptrace[0], ptrace[1], ptrace[2], ptrace[3]);
                }
                *reinterpret_cast<float4*>(gp) = make_float4(th[0], th[1], th[2], th[3]);
            } else if (MODE == MODE_OR) {
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    float hx, hy;
                    unpack2(h[k], hx, hy);
                    if (hx != 0.0f || hy != 0.0f) {                             // R6
                        float t = fmaf(2.0f, fast_atan2_pos(hy, hx), -th[k]);
                        t = (t < 0.0f) ? t + kTwoPiF : t;
                        t = (t >= kTwoPiF) ? t - kTwoPiF : t;
                        th[k] = t;
                    }
                    if (FUSED) {                                                // observables of the NEW state
                        float s, c;
                        fast_sincos(th[k], s, c);
                        accE = fmaf(c, hx, fmaf(s, hy, accE));
                        accM = add2(accM, pack2(c, s));
                    }
                }
                *reinterpret_cast<float4*>(gp) = make_float4(th[0], th[1], th[2], th[3]);
            } else {  // MODE_MEASURE: own = white; E = -sum_white S_i . h_i counts every bond once
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    float hx, hy, s, c;
                    unpack2(h[k], hx, hy);
                    fast_sincos(th[k], s, c);
                    accE = fmaf(c, hx, fmaf(s, hy, accE));
                    accM = add2(accM, pack2(c, s));
                }
            }
        }
        if (MEAS) {
            float mx, my;
            unpack2(accM, mx, my);
            dE += (double)accE; dMx += (double)mx; dMy += (double)my;
            accE = 0.f; accM = 0ull;
        }
    };

    // ---- march: two planes per iteration so that the parity is a compile-time constant ------------
    if (UNI) {
        if (par0) { for (int zi = 0; zi < TZ; zi += 2) { plane(zi, 1); plane(zi + 1, 0); } }
        else      { for (int zi = 0; zi < TZ; zi += 2) { plane(zi, 0); plane(zi + 1, 1); } }
    } else {
        for (int zi = 0; zi < TZ; ++zi) plane(zi, par0 ^ (zi & 1));
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
    if (MEAS) {
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

// Settles the Metropolis decisions the fp32 fast path could not call (|u - p_fast| inside the
// window of xy_device.cuh): the definition of include/xy.h in fp64 from the STORED angles.  Runs
// after each colour pass, before anything reads the updated colour.  Eight lanes share an entry
// (six neighbours, old angle, proposal: one fp64 sincos each).
struct FixupParams {
    float* own; const float* other;
    int L, W, colour, R;
    unsigned int half_n;
    PhiloxKeys keys;
    uint32_t sweep;
    const float* beta32_of_slot;
    unsigned long long* met_acc;
    unsigned long long* exact_count;
    const uint4* near_queue;
    unsigned int* near_count;
    unsigned int near_cap;
    unsigned int* done_ticket;
    unsigned int* overflow_flag;
};

__global__ void __launch_bounds__(256) met_fixup_kernel(const FixupParams F) {
    const unsigned int n_raw = *F.near_count;
    const unsigned int n = n_raw < F.near_cap ? n_raw : F.near_cap;
    const int L = F.L, W = F.W;
    const unsigned int planeG = (unsigned int)L * W;
    const int lane = threadIdx.x & 31, role = lane & 7;
    const unsigned int groups = (gridDim.x * blockDim.x) >> 3;
    const uint32_t stream = F.colour == 0 ? kStreamMetBlack : kStreamMetWhite;
    for (unsigned int e0 = ((blockIdx.x * blockDim.x + threadIdx.x) >> 5) << 2; e0 < n; e0 += groups) {   // warp-uniform trip count
        const unsigned int e = e0 + (lane >> 3);
        const bool live = e < n;
        const uint4 ent = live ? F.near_queue[e] : make_uint4(0u, 0u, 0u, 0u);
        const unsigned int idx = ent.x & 0x7fffffffu;
        const bool fast_acc = (ent.x >> 31) != 0u;
        const int slot = (int)ent.y;
        const float t_old = __uint_as_float(ent.z);
        const int z = (int)(idx / planeG);
        const unsigned int rem = idx - (unsigned int)z * planeG;
        const int y = (int)(rem / (unsigned int)W), xh = (int)(rem - (unsigned int)y * W);
        const int par = (y + z + F.colour) & 1;                     // x parity of this site
        const uint32_t i = (uint32_t)(2 * xh + par) + (uint32_t)L * (uint32_t)(y + L * z);
        uint32_t w[4];
        philox4x32_10(i >> 2, (uint32_t)slot, F.sweep, stream, F.keys, w);
        const int p = (int)((i >> 1) & 1u);
        const float t_new = word_to_angle(p ? w[2] : w[0]);
        const float u = word_to_u24(p ? w[3] : w[1]);
        // neighbours in the order of the definition: -x, -y, -z, +x, +y, +z
        const int xm = par ? xh : (xh == 0 ? W - 1 : xh - 1);
        const int xp = par ? (xh + 1 == W ? 0 : xh + 1) : xh;
        const int ym = y == 0 ? L - 1 : y - 1, yp = y + 1 == L ? 0 : y + 1;
        const int zm = z == 0 ? L - 1 : z - 1, zp = z + 1 == L ? 0 : z + 1;
        const float* __restrict__ other = F.other + (size_t)slot * F.half_n;
        int nx = xh, ny = y, nz = z;
        if (role == 0) nx = xm; else if (role == 1) ny = ym; else if (role == 2) nz = zm;
        else if (role == 3) nx = xp; else if (role == 4) ny = yp; else if (role == 5) nz = zp;
        float a = role == 6 ? t_old : t_new;
        if (role < 6 && live) a = other[((size_t)nz * L + ny) * W + nx];
        double sn_, cs_;
        sincos((double)a, &sn_, &cs_);
        double hx = 0.0, hy = 0.0, co = 0.0, so = 0.0, cn = 0.0, sn = 0.0;
        const int base = lane & ~7;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const double c = __shfl_sync(0xffffffffu, cs_, base + j), s = __shfl_sync(0xffffffffu, sn_, base + j);
            if (j < 6) { hx += c; hy += s; } else if (j == 6) { co = c; so = s; } else { cn = c; sn = s; }
        }
        if (live && role == 0) {
            const double dE = -(hx * (cn - co) + hy * (sn - so));
            const bool acc = (double)u < exp(-(double)F.beta32_of_slot[slot] * dE);
            F.own[(size_t)slot * F.half_n + idx] = acc ? t_new : t_old;
            if (acc != fast_acc) atomicAdd(F.met_acc + slot, acc ? 1ull : ~0ull);
        }
    }
    // the last block to finish resets the queue for the next colour pass
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned int t = atomicAdd(F.done_ticket, 1u);
        if (t == gridDim.x - 1) {
            if (n_raw > F.near_cap) *F.overflow_flag = 1u;
            atomicAdd(F.exact_count, (unsigned long long)n);
            *F.near_count = 0u;
            *F.done_ticket = 0u;
            __threadfence();
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
