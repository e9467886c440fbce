// xy_sweep.cuh -- the colour-pass kernel of the XY Monte Carlo step (sm_100a): Metropolis (a2),
// over-relaxation (a3, optionally carrying the observables) and the standalone reduction (a4).
//
// Data layout in HBM: colour-split, replica-major fp32 angles
//     theta_c[slot][z][y][xh],  c = (x+y+z)&1,  xh = x>>1,  row length W = L/2 floats
// so a colour pass reads both half-lattices once and writes only its own: 12 B per site-update.
//
// A thread block owns a tile of TY full rows of its colour and MARCHES through TZ planes.  Every
// thread owns four consecutive sites (one 128-bit load and store) of one row for the whole march.
// The last warp of the block is an auxiliary warp: its first lane issues the copies, all its lanes
// stage the two halo rows; the other warps all do identical work.
// Raw angles travel HBM -> shared memory as bulk asynchronous copies (TMA, cp.async.bulk) issued
// kRaw-1 steps ahead into a ring of kRaw raw slots, completing on an mbarrier per slot:
// per step the other colour's rows y0-1 .. y0+TY of plane z+1 (three copies: the two halo rows
// wrap in y) and the own colour's TY rows of plane z.  Memory latency is therefore hidden by the
// copy engine, not by registers or occupancy.  Every thread turns the other colour's raw float4 at
// its own (y, x) position into four (cos, sin) pairs ONCE per plane.  Those pairs are exactly the
// z neighbours (planes z-1, z+1) and the x neighbours (plane z) of the thread's own four sites, so it
// keeps them in registers across three steps; shared memory only carries them to the threads of
// the rows above and below (y neighbours) and to the next column (one edge pair), through a ring of
// 3 staged planes.  That halves the shared-memory traffic, which is what bounds this kernel next
// to instruction issue.  The block barrier is split: a thread ARRIVES on an mbarrier right after it
// has staged plane z+1 and only WAITS for that phase at the top of the next step, so warps drift up
// to one plane apart instead of meeting at a __syncthreads per plane.  x wraps inside the tile, y
// and z wrap in the source addresses of the copies.  All per-thread addresses are computed once.
#pragma once
#include <type_traits>
#include "xy_device.cuh"

namespace xyk {

enum { MODE_MET = 0, MODE_OR = 1, MODE_MEASURE = 2, MODE_STIFF = 3 };
constexpr int kRing = 3;                 // staged (cos, sin) planes resident in shared memory
constexpr int kRaw = 6;                  // raw-angle slots filled by bulk copies (a multiple of kRing: see the march)
constexpr int kAhead = 3;                // steps between issuing a copy and reading its slot

struct SweepParams {
    float* own;                  // colour array being updated   [R][L][L][W]
    const float* other;          // the other colour's array (read only during the pass)
    int L, W, W4;                // W = L/2 floats per row, W4 = L/8 float4 per row
    int TY, TZ, nTY, nTZ;        // tile rows, march length, tiles per replica in y and z
    int colour;                  // colour of `own`
    int slot0, n_slots;          // this launch covers the slots [slot0, slot0 + n_slots): blockIdx.y = 0 is slot slot0 (XY_OPT_SLOT_CHUNK)
    int nItems;                  // TY * W4 own float4 per plane (<= blockDim.x)
    unsigned int half_n;         // L^3 / 2 floats per slot per colour
    PhiloxKeys keys;
    uint32_t sweep;              // n_met (Philox counter word 2) ...
    const uint32_t* d_counters;  // ... or, when not null, read from d_counters[0] (CUDA-graph replay: see DeviceCounters)
    const float* beta32_of_slot; // Metropolis: fp32 beta label per slot (R13)
    unsigned long long* met_acc; // Metropolis: accepted proposals per slot
    unsigned long long* exact_count;  // Metropolis: decisions re-evaluated in fp64
    float* trace;                // Metropolis test hook: p_fast per own site (same layout as own) or null
    double* partials;            // measure: [R][nTY*nTZ][3] partial E, Mx, My; MODE_STIFF: [R][nTY*nTZ][6] Cx,Cy,Cz,Sx,Sy,Sz
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
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
// ---- mbarrier (shared::cta): the split arrive / wait block barrier -------------------------------
__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// try_wait suspends the thread until the phase completes or the time hint (ns) expires
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n .reg .pred p;\n"
        "XY_WAIT:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"
        " @p bra XY_DONE;\n bra XY_WAIT;\n"
        "XY_DONE:\n}" ::"r"(bar), "r"(parity), "r"(1000000u) : "memory");
}

// ---- shared-memory accesses by 32-bit shared-window address (keeps every address a single register
//      plus an immediate) --------------------------------------------------------------------------
__device__ __forceinline__ float4 lds_f4(uint32_t a) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}
__device__ __forceinline__ ulonglong2 lds_p2(uint32_t a) {        // two (cos, sin) pairs
    ulonglong2 v;
    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(v.x), "=l"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ f32x2 lds_p1(uint32_t a) {
    f32x2 v;
    asm volatile("ld.shared.b64 %0, [%1];" : "=l"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts_f4(uint32_t a, float x, float y, float z, float w) {
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(a), "f"(x), "f"(y), "f"(z), "f"(w) : "memory");
}
// Loop-invariant per-thread values pass through this so that the compiler keeps them in a register
// instead of recomputing them from the thread index on every step of the march.
__device__ __forceinline__ void keep(uint32_t& x) { asm volatile("" : "+r"(x)); }
__device__ __forceinline__ void keep(int& x) { asm volatile("" : "+r"(x)); }
__device__ __forceinline__ void keep(float& x) { asm volatile("" : "+f"(x)); }

// Appends one close Metropolis decision to the queue settled by met_fixup_kernel (rare path).
__device__ __noinline__ void push_near(unsigned int* near_count, uint4* near_queue, unsigned int near_cap,
                                       unsigned int idx_acc, unsigned int slot, float t_old) {
    const unsigned int e = atomicAdd(near_count, 1u);
    if (e < near_cap) near_queue[e] = make_uint4(idx_acc, slot, __float_as_uint(t_old), 0u);
}

// ---- TMA bulk copy global -> shared, completing on an mbarrier ----------------------------------------
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}


// Padding of a staged row (bytes, a multiple of 16).  A warp's 128-bit accesses to a staged row go to consecutive
// 16-byte words, eight lanes per wavefront; where a warp continues in its NEXT row (the row `jump` staged rows further:
// 1 in the row-major thread mapping, 2 where the warps are mapped to rows of one parity), the eight lanes around the
// break still hit eight different bank groups only if that row starts where this one's part ended, modulo the 128
// bytes of the banks:  jump * (W4*32 + pad) == W4*16  (mod 128).  Without padding this fails whenever W4 is not a
// multiple of 8 (L = 160: W4 = 20, 3.3e6 + 1.9e6 excess wavefronts per launch on the loads of the rows above / below
// and on the staging stores; profiles/r3_head.md).  0 where no multiple of 16 solves it or XY_STAGE_PAD is 0.
#ifndef XY_STAGE_PAD
#define XY_STAGE_PAD 1
#endif
__host__ __device__ constexpr int stage_pad_bytes(int W4, bool uni) {
    if (!XY_STAGE_PAD) return 0;
    for (int pad = 0; pad < 128; pad += 16)
        if (((uni ? 2 : 1) * (W4 * 32 + pad) - W4 * 16) % 128 == 0) return pad;
    return 0;
}

// Shared memory of one block (bytes):  kRing staged planes of (TY+2) rows x (W pairs x 8 + padding)  |
// kRaw raw slots of (2 TY + 2) rows x W floats x 4 (other colour first, then own)  |  1 + kRaw mbarriers
// uni: the warps of the kernel variant are mapped to rows of one parity (compile-time geometry, see sweep_kernel)
__host__ __device__ inline size_t sweep_smem_bytes(int L, int TY, bool uni = false) {
    return (size_t)kRing * (TY + 2) * ((L / 2) * 8 + stage_pad_bytes(L / 8, uni)) + (size_t)kRaw * (2 * TY + 2) * (L / 2) * 4 + 8 * (1 + kRaw) + 8;
}
// the larger of the two mappings' needs (tile validation on the host, before a kernel variant is chosen)
__host__ __device__ inline size_t sweep_smem_bytes_max(int L, int TY) {
    const size_t a = sweep_smem_bytes(L, TY, false), b = sweep_smem_bytes(L, TY, true);
    return a > b ? a : b;
}

// W4C, TYC: L/8 and the tile rows as compile-time constants (every shared-memory pitch becomes an
// immediate; where TYC*W4C/2 is a multiple of 32 the warps are mapped to rows of one parity, so that the
// x parity of a warp's sites is uniform), or 0, 0 = read the geometry from P, any tile.
// EXACT_INLINE (Metropolis only): re-evaluate close decisions in fp64 on the spot (function call in
// the loop: slow; chosen by the launcher when |beta| is so large that most decisions are "close").
// Otherwise close decisions are appended to a global queue and settled by met_fixup_kernel, which
// keeps the fp64 code and its registers out of this loop.
#ifndef XY_SWEEP_MIN_BLOCKS
#define XY_SWEEP_MIN_BLOCKS 2
#endif
#ifndef XY_MET_EARLY_DRAW
#define XY_MET_EARLY_DRAW 1
#endif
template <int MODE, bool TRACE, bool FUSED, bool EXACT_INLINE, int W4C, int TYC, bool PDL = false>
__global__ void __launch_bounds__(W4C ? (W4C * TYC + 31) / 32 * 32 + 32 : 384, (W4C * TYC > 352) ? 1 : XY_SWEEP_MIN_BLOCKS) sweep_kernel(const SweepParams P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr bool UNI = W4C != 0 && (W4C * TYC / 2) % 32 == 0;   // whole warps per row parity (L = 80: compile-time geometry only)
    const int L = P.L;
    const int W4 = W4C ? W4C : P.W4;
    const int W = 4 * W4;
    const int TY = TYC ? TYC : P.TY, TZ = P.TZ;
    const int rowB = W * 8 + stage_pad_bytes(W4, UNI);   // bytes per staged row (W pairs + bank padding)
    const int partB = W4 * 16;                       // byte offset of part B inside a row
    const int planeB = (TY + 2) * rowB;              // bytes per staged plane; ring of kRing planes
    const int ringB = kRing * planeB;
    const int rawRowB = W * 4;                       // bytes per raw row
    const int rawOwnB = (TY + 2) * rawRowB;          // own rows follow the other colour's TY+2 rows
    const int rawSlotB = (2 * TY + 2) * rawRowB;
    const uint32_t sm0 = smem_addr(smem_raw);        // staged ring
    const uint32_t raw0 = sm0 + ringB;               // raw slots
    const uint32_t bar = raw0 + kRaw * rawSlotB;     // step barrier, then kRaw "slot full" barriers
    const uint32_t full0 = bar + 8;

    const int tid = threadIdx.x;
    const int slot = blockIdx.y + P.slot0;
    const int tile = blockIdx.x;
    const int tzi = tile / P.nTY, tyi = tile - tzi * P.nTY;
    const int y0 = tyi * TY, z0 = tzi * TZ;
    const int nSteps = TZ + 2;                       // step s stages plane s-1 (relative to z0) and updates plane s-2
    const int nCompute = (int)blockDim.x - 32;       // the last warp is the auxiliary warp

    const float* __restrict__ other = P.other + (size_t)slot * P.half_n;
    float* __restrict__ own = P.own + (size_t)slot * P.half_n;
    const unsigned int planeG = (unsigned int)L * W;

    if (tid == 0) {
        mbar_init(bar, blockDim.x);
        for (int k = 0; k < kRaw; ++k) mbar_init(full0 + 8 * k, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // everything above touched shared memory only; from here on the kernel reads what its predecessor wrote
    // PDL: this instantiation is launched with programmatic stream serialization (xy_device.cuh).  A template parameter,
    // not a run-time flag: the mere presence of the two instructions cost the over-relaxation pass 0.2-0.3 % at
    // L = 160 x 64, where the launcher does not use them (profiles/r3_experiments.md)
    if (PDL) {
        allow_dependent_launch();
        grid_dependency_wait();
    }

    constexpr bool MEAS = (MODE == MODE_MEASURE) || FUSED;
    constexpr bool STIFF = MODE == MODE_STIFF;          // the six bond sums of Eq. 6 instead of E, Mx, My
    float acc6[6] = { 0.f, 0.f, 0.f, 0.f, 0.f, 0.f };
    double d6[6] = { 0.0, 0.0, 0.0, 0.0, 0.0, 0.0 };
    f32x2 accM = 0ull;                               // per-plane fp32 (Mx, My), flushed to double each plane
    f32x2 accE = 0ull;                               // (sum cos_i h_x, sum sin_i h_y): E = -(x + y)
    double dE = 0.0, dMx = 0.0, dMy = 0.0;
    unsigned int nacc = 0, nexact = 0;
    bool active = false;

    // raw float4 at `src` -> (cos, sin) of its four angles -> registers pp[] and staged plane at `dst`
    auto stage = [&](uint32_t src, uint32_t dst, f32x2 (&pp)[4]) {
        const float4 v = lds_f4(src);
        float c0, s0, c1, s1, c2, s2, c3, s3;
        fast_sincos(v.x, s0, c0); fast_sincos(v.y, s1, c1);
        fast_sincos(v.z, s2, c2); fast_sincos(v.w, s3, c3);
        sts_f4(dst, c0, s0, c1, s1);
        sts_f4(dst + partB, c2, s2, c3, s3);
        pp[0] = pack2(c0, s0); pp[1] = pack2(c1, s1); pp[2] = pack2(c2, s2); pp[3] = pack2(c3, s3);
    };

    // Phase s of the step barrier completes when every thread has arrived s+1 times: once before the
    // march, then once per step after its staging and raw reads.  Waiting for phase s at the top of
    // step s therefore means: every thread has staged plane s-2 (the one whose rows this step reads),
    // has finished updating plane s-4 (ring slot s % kRing is free) and has read raw slot
    // (s-1) % kRaw (free for the next copies).
    int sS = 0;                                      // ring byte offset of the plane staged this step (slot s % kRing)
    int rS = 0;                                      // raw byte offset of this step's slot (s % kRaw)
    uint32_t fullBar = full0;                        // this step's "slot full" barrier and the parity of its phase
    uint32_t fullPar = 0;
    auto advance = [&]() {
        sS += planeB; if (sS == ringB) sS = 0;
        rS += rawSlotB; fullBar += 8;
        if (rS == kRaw * rawSlotB) { rS = 0; fullBar = full0; fullPar ^= 1u; }
    };

    if (tid >= nCompute) {
        // ---- auxiliary warp: bulk copies (lane 0) and the halo rows y0-1, y0+TY of every staged plane ----
        const int lane = tid - nCompute;
        int ylo = y0 - 1, yhi = y0 + TY;
        if (ylo < 0) ylo += L;
        if (yhi >= L) yhi -= L;
        auto issue = [&](int s) {                    // fill raw slot s % kRaw for step s
            const int rs = s % kRaw;
            const uint32_t fb = full0 + 8 * rs;
            const uint32_t dst = raw0 + rs * rawSlotB;
            const bool has_other = true, has_own = s >= 2;
            mbar_expect_tx(fb, (has_other ? (TY + 2) * rawRowB : 0) + (has_own ? TY * rawRowB : 0));
            if (has_other) {
                int z = z0 + s - 1; if (z < 0) z += L; if (z >= L) z -= L;
                const float* pl = other + (size_t)z * planeG;
                bulk_g2s(dst, pl + (size_t)ylo * W, rawRowB, fb);
                bulk_g2s(dst + rawRowB, pl + (size_t)y0 * W, TY * rawRowB, fb);
                bulk_g2s(dst + (TY + 1) * rawRowB, pl + (size_t)yhi * W, rawRowB, fb);
            }
            if (has_own) bulk_g2s(dst + rawOwnB, own + (size_t)(z0 + s - 2) * planeG + (size_t)y0 * W, TY * rawRowB, fb);
        };
        if (lane == 0)
            for (int s = 0; s < kAhead && s < nSteps; ++s) issue(s);
        mbar_arrive(bar);
#pragma unroll 1
        for (int s = 0; s < nSteps; ++s) {
            mbar_wait(bar, (uint32_t)s & 1u);
            mbar_wait(fullBar, fullPar);
            for (int j = lane; j < 2 * W4; j += 32) {
                const int r2 = j >= W4, q2 = j - (r2 ? W4 : 0);
                f32x2 pp[4];
                stage(raw0 + rS + ((r2 ? TY + 1 : 0) * W + 4 * q2) * 4, sm0 + sS + (r2 ? TY + 1 : 0) * rowB + q2 * 16, pp);
            }
            mbar_arrive(bar);                        // the compute warps wait for this: copies come after it
            if (lane == 0 && s + kAhead < nSteps) issue(s + kAhead);
            advance();
        }
    } else {
        // ---- compute warps.  This thread's own item: row ty of the tile, float4 column q; idle threads
        //      (compute threads rounded up to a warp) shadow item 0 and store nothing.  UNI: warps
        //      [0, n/2) take the even rows, the rest the odd rows, so the x parity is uniform over a warp
        active = (W4C != 0 && (W4C * TYC) % 32 == 0) || tid < P.nItems;
        const int item = active ? tid : 0;
        int ty, q;
        if (UNI) {
            constexpr int half = W4C * TYC / 2;
            const int cls = item >= half;
            const int r = item - (cls ? half : 0);
            const int t2 = r / W4;
            ty = 2 * t2 + cls; q = r - t2 * W4;
        } else {
            ty = item / W4; q = item - ty * W4;
        }
        const int y = y0 + ty;
        // Staged plane: (TY+2) rows.  A row of W = 4*W4 sites is stored as two arrays of W4 x 16 bytes:
        // part A holds the (cos, sin) pairs of sites 4q, 4q+1, part B those of sites 4q+2, 4q+3, so
        // that consecutive lanes read consecutive 16-byte words (no bank conflicts) and a thread's four
        // sites are two 128-bit loads.  This thread stages the other colour's float4 at its own (y, q).
        uint32_t aRow = sm0 + (ty + 1) * rowB + q * 16;              // staged row ty+1, part A, column q (+ ring offset)
        uint32_t aRawO = raw0 + ((ty + 1) * W + 4 * q) * 4;          // raw other-colour float4 (+ raw slot offset);
        const int ownDelta = rawOwnB - rawRowB;                      // the raw own-colour float4 sits this much further
        // edge pair of the row: par = 0 needs site 4q-1 (part B of column q-1, second pair),
        // par = 1 needs site 4q+4 (part A of column q+1, first pair); x wraps inside the row.
        int eRel0 = partB + ((q == 0 ? W4 - 1 : q - 1) - q) * 16 + 8;            // relative to aRow
        int eRel1 = ((q + 1 == W4 ? 0 : q + 1) - q) * 16;
        // x parity of this row's own sites on plane z: (y + z + colour) & 1; flips every plane
        int par = (y + z0 + P.colour) & 1;
        // Philox counter word 0 of this thread's first quad on plane z0; a plane further is +L*L/4
        uint32_t ctr0 = (uint32_t)(2 * q) + (uint32_t)(L >> 2) * (uint32_t)(y + L * z0);
        const uint32_t ctrStep = (uint32_t)(L >> 2) * (uint32_t)L;
        unsigned int gz = (unsigned int)z0 * planeG + (unsigned int)y * W + 4 * q;   // element index of the own float4 being updated
        float* gp = own + gz;                                                        // and its address
        keep(aRow); keep(aRawO); keep(eRel0); keep(eRel1); keep(par); keep(ctr0);

        float bl = 0.f, win24 = 0.f, beta32 = 0.f;
        PhiloxInv inv = {0u, 0u, 0u, 0u};
        if (MODE == MODE_MET) {
            beta32 = P.beta32_of_slot[slot];
            bl = beta32 * 1.44269504f;               // exp(beta g) = 2^(bl g)
            win24 = (fabsf(beta32) * kWindowPerBeta + kWindowAbs) * 4294967296.0f;  // window in units of 2^-32, see xy_device.cuh
            inv = philox_block_invariants((uint32_t)slot, P.d_counters ? P.d_counters[0] : P.sweep, P.colour == 0 ? kStreamMetBlack : kStreamMetWhite, P.keys);
            keep(bl); keep(win24); keep(inv.j0); keep(inv.j1); keep(inv.j2); keep(inv.j3);
        }
        // (cos, sin) pairs of the other colour at this thread's own (y, x) position on three consecutive
        // planes; the roles (z-1, z, z+1) rotate from step to step, so the march is unrolled by three
        // (J = s % 3 at compile time: staged-ring slot, raw slot J or J+3, and the roles are all static)
        f32x2 P0[4] = {0ull, 0ull, 0ull, 0ull}, P1[4] = {0ull, 0ull, 0ull, 0ull}, P2[4] = {0ull, 0ull, 0ull, 0ull};
        int rH = 0;                                  // 0: raw slots 0..2, 1: raw slots 3..5 (toggles every three steps)

        auto step = [&](const int s, auto do_update, auto jc, f32x2 (&pm)[4], f32x2 (&pc)[4], f32x2 (&pp)[4]) {
            constexpr bool UPDATE = decltype(do_update)::value;
            constexpr int J = decltype(jc)::value;
            if (J == 0 && s > 0) { rH ^= 1; if (!rH) fullPar ^= 1u; }
            const uint32_t aS = aRow + J * planeB, aZ = aRow + ((J + 2) % 3) * planeB;   // planes z+1 (staged now) and z
            mbar_wait(bar, (uint32_t)s & 1u);
            mbar_wait(full0 + 8 * J + (rH ? 24 : 0), fullPar);       // this step's raw rows have landed
            const uint32_t rO = aRawO + J * rawSlotB + (rH ? 3 * rawSlotB : 0);
            float4 cur = make_float4(0.f, 0.f, 0.f, 0.f);
            // Metropolis (XY_MET_EARLY_DRAW): this plane's random words are drawn while the plane is staged, the two
            // Philox calls advanced round by round side by side, so that ptxas interleaves their multiply -> xor
            // chains (four independent multiplies per round instead of two) and overlaps them with the shared-memory
            // loads and the field sums that follow.  Measured at L=160: -1.2 % per pass; pinning the sin/cos of the
            // old angles up here as well (volatile asm, or dependencies through an opaque zero) cost registers
            // (spills under the 80-register cap) and 7 %.
            constexpr bool EARLY = XY_MET_EARLY_DRAW && MODE == MODE_MET && UPDATE;
            uint32_t wq[2][4] = { {0u, 0u, 0u, 0u}, {0u, 0u, 0u, 0u} };
            if (EARLY) {
                stage(rO, aS, pp);
                cur = lds_f4(rO + ownDelta);
                PhiloxState A, B;
                philox_var0_start(ctr0, inv, P.keys, A);
                philox_var0_start(ctr0 + 1u, inv, P.keys, B);
                philox_round<3>(A, P.keys); philox_round<3>(B, P.keys);
                philox_round<4>(A, P.keys); philox_round<4>(B, P.keys);
                philox_round<5>(A, P.keys); philox_round<5>(B, P.keys);
                mbar_arrive(bar);
                philox_round<6>(A, P.keys); philox_round<6>(B, P.keys);
                philox_round<7>(A, P.keys); philox_round<7>(B, P.keys);
                philox_round<8>(A, P.keys); philox_round<8>(B, P.keys);
                philox_round<9>(A, P.keys); philox_round<9>(B, P.keys);
                wq[0][0] = A.c0; wq[0][1] = A.c1; wq[0][2] = A.c2; wq[0][3] = A.c3;
                wq[1][0] = B.c0; wq[1][1] = B.c1; wq[1][2] = B.c2; wq[1][3] = B.c3;
            } else {
                stage(rO, aS, pp);
                if (MEAS && active && s >= 1 && s <= TZ) accM = add2(accM, add2(add2(pp[0], pp[1]), add2(pp[2], pp[3])));
                if (UPDATE) cur = lds_f4(rO + ownDelta);
                mbar_arrive(bar);
            }
            if (UPDATE) {
                // ---- local fields of the four own sites: z neighbours and the row itself from registers,
                //      y neighbours (rows above and below) and the edge pair from the staged plane z ------
                f32x2 h[4];
                {
                    const f32x2 e = lds_p1(aZ + (par ? eRel1 : eRel0));
                    const ulonglong2 aA = lds_p2(aZ - rowB), aB = lds_p2(aZ - rowB + partB);
                    const ulonglong2 bA = lds_p2(aZ + rowB), bB = lds_p2(aZ + rowB + partB);
                    if (STIFF) {
                        // Per direction mu and own (white) site i the two bonds (i-mu, i) and (i, i+mu):
                        //   C_mu += S_i . (S_- + S_+),   S_mu += sin_i (cos_+ - cos_-) - cos_i (sin_+ - sin_-);
                        // the white sites' bonds are all bonds (bipartite lattice).  Not a hot path: scalar fp32.
                        const f32x2 ym[4] = { aA.x, aA.y, aB.x, aB.y }, yp[4] = { bA.x, bA.y, bB.x, bB.y };
                        const float own4[4] = { cur.x, cur.y, cur.z, cur.w };
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            const f32x2 xm = par ? pc[k] : (k == 0 ? e : pc[k - 1]);
                            const f32x2 xp = par ? (k == 3 ? e : pc[k + 1]) : pc[k];
                            const f32x2 lo[3] = { xm, ym[k], pm[k] }, hi[3] = { xp, yp[k], pp[k] };
                            float si, ci;
                            fast_sincos(own4[k], si, ci);
#pragma unroll
                            for (int mu = 0; mu < 3; ++mu) {
                                float cm, sm, cp, sp;
                                unpack2(lo[mu], cm, sm); unpack2(hi[mu], cp, sp);
                                acc6[mu] = fmaf(ci, cm + cp, fmaf(si, sm + sp, acc6[mu]));
                                acc6[3 + mu] = fmaf(si, cp - cm, fmaf(-ci, sp - sm, acc6[3 + mu]));
                            }
                        }
                    }
                    const f32x2 y0s = add2(add2(aA.x, bA.x), add2(pm[0], pp[0]));
                    const f32x2 y1s = add2(add2(aA.y, bA.y), add2(pm[1], pp[1]));
                    const f32x2 y2s = add2(add2(aB.x, bB.x), add2(pm[2], pp[2]));
                    const f32x2 y3s = add2(add2(aB.y, bB.y), add2(pm[3], pp[3]));
                    // x neighbours: par = 0 -> sites (j-1, j), par = 1 -> sites (j, j+1) of the same row
                    const f32x2 s01 = add2(pc[0], pc[1]), s12 = add2(pc[1], pc[2]), s23 = add2(pc[2], pc[3]);
                    if (UNI) {                       // warp-uniform branch
                        if (par) { h[0] = add2(y0s, s01); h[1] = add2(y1s, s12); h[2] = add2(y2s, s23); h[3] = add2(y3s, add2(pc[3], e)); }
                        else     { h[0] = add2(y0s, add2(e, pc[0])); h[1] = add2(y1s, s01); h[2] = add2(y2s, s12); h[3] = add2(y3s, s23); }
                    } else {
                        const f32x2 se = add2(e, par ? pc[3] : pc[0]);
                        h[0] = add2(y0s, par ? s01 : se); h[1] = add2(y1s, par ? s12 : s01);
                        h[2] = add2(y2s, par ? s23 : s12); h[3] = add2(y3s, par ? se : s23);
                    }
                }
                float th[4] = { cur.x, cur.y, cur.z, cur.w };

                if (MODE == MODE_MET) {
                    float ptrace[4], dist[4];
#pragma unroll
                    for (int pr = 0; pr < 2; ++pr) {
                        uint32_t w[4];
                        if (EARLY) { w[0] = wq[pr][0]; w[1] = wq[pr][1]; w[2] = wq[pr][2]; w[3] = wq[pr][3]; }
                        else philox4x32_10_var0(ctr0 + pr, inv, P.keys, w);
#pragma unroll
                        for (int kk = 0; kk < 2; ++kk) {
                            const int k = 2 * pr + kk;
                            const float kf = (float)(w[2 * kk] >> 8);
                            const float tn = kf * kTwoPiU24;
                            // acceptance uniform, fast path: the whole word converted in ONE instruction (2^32 u24 up
                            // to the rounding of its low byte, < 2^-24 absolute, which kWindowAbs covers)
                            const float uf = (float)w[2 * kk + 1];
                            float hx, hy, so, co, sn, cn;
                            unpack2(h[k], hx, hy);
                            fast_sincos(th[k], so, co);
                            fast_sincos(tn, sn, cn);
                            const float g = fmaf(hx, cn - co, hy * (sn - so));   // = -dE
                            const float pf = fast_ex2(fmaf(bl, g, 32.0f));        // p * 2^32
                            bool acc = uf < pf;
                            dist[k] = fabsf(uf - pf);
                            if (EXACT_INLINE && dist[k] < win24) {
                                acc = metropolis_exact(other, L, W, par, 4 * q + k, y, z0 + s - 2, th[k], tn, word_to_u24(w[2 * kk + 1]), beta32);
                                ++nexact;
                            }
                            if (TRACE) ptrace[k] = fminf(pf * 2.3283064365386963e-10f, 3.0e38f);
                            if (acc) { th[k] = tn; ++nacc; }
                        }
                    }
                    // decisions too close to call in fp32: queue them for met_fixup_kernel (rare)
                    if (!EXACT_INLINE && fminf(fminf(dist[0], dist[1]), fminf(dist[2], dist[3])) < win24 && active) {
                        const float old[4] = { cur.x, cur.y, cur.z, cur.w };
#pragma unroll
                        for (int k = 0; k < 4; ++k)
                            if (dist[k] < win24) {
                                const bool fast_acc = __float_as_uint(th[k]) != __float_as_uint(old[k]);
                                push_near(P.near_count, P.near_queue, P.near_cap, (gz + k) | (fast_acc ? 0x80000000u : 0u),
                                          (unsigned int)slot, old[k]);
                            }
                    }
                    if (TRACE && active) {
                        float* tr = P.trace + (size_t)P.colour * gridDim.y * P.half_n + (size_t)slot * P.half_n;
                        *reinterpret_cast<float4*>(tr + gz) = make_float4(ptrace[0], ptrace[1], ptrace[2], ptrace[3]);
                    }
                    ctr0 += ctrStep;
                } else if (MODE == MODE_OR) {
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        float hx, hy;
                        unpack2(h[k], hx, hy);
                        // branch-free so that the four sites' dependency chains interleave; h = 0 gives
                        // NaN through rcp(0) * 0, which the final select discards (R6: spin unchanged)
                        float t = fmaf(2.0f, fast_atan2_pos(hy, hx), -th[k]);
                        t = (t < 0.0f) ? t + kTwoPiF : t;
                        t = (t >= kTwoPiF) ? t - kTwoPiF : t;
                        th[k] = (fmaxf(fabsf(hx), fabsf(hy)) > 0.0f) ? t : th[k];
                        if (FUSED) {                                            // observables of the NEW state
                            float sn, cs;
                            fast_sincos(th[k], sn, cs);
                            const f32x2 sp = pack2(cs, sn);
                            accE = fma2(sp, h[k], accE);
                            accM = add2(accM, sp);
                        }
                    }
                } else if (MODE == MODE_MEASURE) {  // own = white; E = -sum_white S_i . h_i counts every bond once
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        float sn, cs;
                        fast_sincos(th[k], sn, cs);
                        const f32x2 sp = pack2(cs, sn);
                        accE = fma2(sp, h[k], accE);
                        accM = add2(accM, sp);
                    }
                }
                if (MODE != MODE_MEASURE && !STIFF && active) *reinterpret_cast<float4*>(gp) = make_float4(th[0], th[1], th[2], th[3]);
                if (STIFF) {
#pragma unroll
                    for (int c = 0; c < 6; ++c) { if (active) d6[c] += (double)acc6[c]; acc6[c] = 0.f; }
                }
                // fp32 partial sums go to the fp64 accumulators once per unrolled triple of steps (at most 24
                // terms of magnitude <= 6 each in fp32: 1e-5 absolute per flush, far below the 1e-6 * 3N bar)
                if (MEAS && (J == 1 || s == nSteps - 1)) {
                    float mx, my, ex, ey;
                    unpack2(accM, mx, my);
                    unpack2(accE, ex, ey);
                    if (active) { dE += (double)(ex + ey); dMx += (double)mx; dMy += (double)my; }
                    accE = 0ull; accM = 0ull;
                }
                gz += planeG;
                gp += planeG;
                par ^= 1;
            }
        };

        // ---- the march: steps 0 and 1 only stage planes -1 and 0; step s stages into P[s % 3] ------------
        mbar_arrive(bar);
        using T = std::true_type; using F = std::false_type;
        using J0 = std::integral_constant<int, 0>; using J1 = std::integral_constant<int, 1>; using J2 = std::integral_constant<int, 2>;
        step(0, F{}, J0{}, P1, P2, P0);
        step(1, F{}, J1{}, P2, P0, P1);
        int s = 2;
#pragma unroll 1
        for (; s + 3 <= nSteps; s += 3) {
            step(s, T{}, J2{}, P0, P1, P2);
            step(s + 1, T{}, J0{}, P1, P2, P0);
            step(s + 2, T{}, J1{}, P2, P0, P1);
        }
        if (s < nSteps) { step(s, T{}, J2{}, P0, P1, P2); ++s; }
        if (s < nSteps) { step(s, T{}, J0{}, P1, P2, P0); ++s; }
    }

    // ---- epilogue ---------------------------------------------------------------------------
    if (MODE == MODE_MET) {
        unsigned int a = active ? nacc : 0u, e = active ? nexact : 0u;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, o); e += __shfl_xor_sync(0xffffffffu, e, o); }
        if ((tid & 31) == 0) {
            if (a) atomicAdd(P.met_acc + slot, (unsigned long long)a);
            if (e) atomicAdd(P.exact_count, (unsigned long long)e);
        }
    }
    if (MEAS || STIFF) {
        // fixed-order block reduction in double: warp shuffle tree, then warp 0 sums the warps in order
        constexpr int NV = STIFF ? 6 : 3;
        __shared__ double red[NV][32];
        double v[6] = { STIFF ? d6[0] : dE, STIFF ? d6[1] : dMx, STIFF ? d6[2] : dMy, d6[3], d6[4], d6[5] };
#pragma unroll
        for (int c = 0; c < NV; ++c)
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v[c] += __shfl_xor_sync(0xffffffffu, v[c], o);
        const int wid = tid >> 5, nw = (blockDim.x + 31) >> 5;
        if ((tid & 31) == 0) {
#pragma unroll
            for (int c = 0; c < NV; ++c) red[c][wid] = v[c];
        }
        __syncthreads();
        if (tid < NV) {
            double sum = 0.0;
            for (int k = 0; k < nw; ++k) sum += red[tid][k];
            P.partials[((size_t)slot * gridDim.x + tile) * NV + tid] = (!STIFF && tid == 0) ? -sum : sum;
        }
    }
}

}  // namespace xyk
