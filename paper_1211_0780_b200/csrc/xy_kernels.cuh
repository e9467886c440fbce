// xy_kernels.cuh -- the small kernels of the XY Monte Carlo step (sm_100a): fp64 settlement of close
// Metropolis decisions, final reduction stage, replica exchange, start states, layout conversion
// and the device-math test hooks.  The colour-pass kernel itself is in xy_sweep.cuh.
#pragma once
#include "xy_device.cuh"
#include "xy_sweep.cuh"

namespace xyk {

// Settles the Metropolis decisions the fp32 fast path could not call (|u - p_fast| inside the
// window of xy_device.cuh): the definition of include/xy.h in fp64 from the STORED angles.  Runs
// after each colour pass, before anything reads the updated colour.  Eight lanes share an entry
// (six neighbours, old angle, proposal: one fp64 sincos each).
// Counters of a Monte Carlo step kept on the device so that ONE captured CUDA graph of a step can be
// replayed: the Metropolis kernels read n_met, finalize_pt_kernel reads n_pt and the series row and
// advances everything at the end of the step.
struct DeviceCounters { uint32_t n_met, n_or, n_pt, row; double* series_base; };

__global__ void set_device_counters_kernel(DeviceCounters* dc, DeviceCounters v) { *dc = v; }

struct FixupParams {
    float* own; const float* other;
    int L, W, colour, R;
    unsigned int half_n;
    PhiloxKeys keys;
    uint32_t sweep;
    const uint32_t* d_counters;      // when not null: sweep = d_counters[0] (CUDA-graph replay)
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
    allow_dependent_launch();
    grid_dependency_wait();                      // the colour pass that filled the queue has completed
    const unsigned int n_raw = *F.near_count;
    const unsigned int n = n_raw < F.near_cap ? n_raw : F.near_cap;
    const int L = F.L, W = F.W;
    const unsigned int planeG = (unsigned int)L * W;
    const int lane = threadIdx.x & 31, role = lane & 7;
    const unsigned int groups = (gridDim.x * blockDim.x) >> 3;
    const uint32_t stream = F.colour == 0 ? kStreamMetBlack : kStreamMetWhite;
    const uint32_t sweep = F.d_counters ? F.d_counters[0] : F.sweep;
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
        philox4x32_10(i >> 2, (uint32_t)slot, sweep, stream, F.keys, w);
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
        sincos_0_2pi((double)a, sn_, cs_);
        const double lu = accept_log_u((double)u);
        double hx = 0.0, hy = 0.0, co = 0.0, so = 0.0, cn = 0.0, sn = 0.0;
        const int base = lane & ~7;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const double c = __shfl_sync(0xffffffffu, cs_, base + j), s = __shfl_sync(0xffffffffu, sn_, base + j);
            if (j < 6) { hx += c; hy += s; } else if (j == 6) { co = c; so = s; } else { cn = c; sn = s; }
        }
        if (live && role == 0) {
            const double dE = -(hx * (cn - co) + hy * (sn - so));
            const bool acc = accept_exact((double)u, lu, -(double)F.beta32_of_slot[slot] * dE);
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

// Final stage of a4, shared by the two kernels below: one WARP sums the tile partials of one slot in
// fixed order (lane l takes tiles l, l+32, ..., then a shuffle tree) and lane 0 writes the five
// observables by rank and by slot.
__device__ __forceinline__ void finalize_rank(const double* __restrict__ partials, int n_tiles, int k, int slot, int lane,
                                              double* __restrict__ obs_rank, double* __restrict__ obs_slot,
                                              double* __restrict__ series_row) {
    double v[3] = { 0.0, 0.0, 0.0 };
    for (int t = lane; t < n_tiles; t += 32)
        for (int c = 0; c < 3; ++c) v[c] += partials[((size_t)slot * n_tiles + t) * 3 + c];
    for (int c = 0; c < 3; ++c)
        for (int o = 16; o > 0; o >>= 1) v[c] += __shfl_xor_sync(0xffffffffu, v[c], o);
    if (lane == 0) {
        const double m2 = v[1] * v[1] + v[2] * v[2];
        const double o5[5] = { v[0], v[1], v[2], m2, m2 * m2 };
        for (int c = 0; c < 5; ++c) {
            obs_rank[5 * k + c] = o5[c];
            obs_slot[5 * slot + c] = o5[c];
            if (series_row) series_row[5 * k + c] = o5[c];
        }
    }
}

// grid: one warp per rank
__global__ void measure_finalize_kernel(const double* __restrict__ partials, int n_tiles, int R,
                                        const int* __restrict__ slot_at_rank,
                                        double* __restrict__ obs_rank, double* __restrict__ obs_slot,
                                        double* __restrict__ series_row) {
    const int k = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (k < R) finalize_rank(partials, n_tiles, k, slot_at_rank[k], threadIdx.x & 31, obs_rank, obs_slot, series_row);
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

// Final stage of the six spin-stiffness sums: one warp per rank, fixed order.
__global__ void stiffness_finalize_kernel(const double* __restrict__ partials6, int n_tiles, int R,
                                          const int* __restrict__ slot_at_rank, double* __restrict__ out6_rank) {
    const int k = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (k >= R) return;
    const int slot = slot_at_rank[k];
    double v[6] = { 0.0, 0.0, 0.0, 0.0, 0.0, 0.0 };
    for (int t = lane; t < n_tiles; t += 32)
        for (int c = 0; c < 6; ++c) v[c] += partials6[((size_t)slot * n_tiles + t) * 6 + c];
    for (int c = 0; c < 6; ++c)
        for (int o = 16; o > 0; o >>= 1) v[c] += __shfl_xor_sync(0xffffffffu, v[c], o);
    if (lane == 0)
        for (int c = 0; c < 6; ++c) out6_rank[6 * k + c] = v[c];
}

// a4 final stage + a5 in one launch (the Monte Carlo step's tail): the 32 warps of one block reduce
// the ranks w, w+32, ... exactly like measure_finalize_kernel, then the block decides the exchanges.
__global__ void __launch_bounds__(1024) finalize_pt_kernel(const double* __restrict__ partials, int n_tiles, int R, uint32_t n_pt,
                                                          PhiloxKeys keys, const double* __restrict__ betas,
                                                          int* __restrict__ slot_at_rank, double* __restrict__ obs_rank,
                                                          double* __restrict__ obs_slot, double* __restrict__ series_row,
                                                          double* __restrict__ beta_of_slot, float* __restrict__ beta32_of_slot,
                                                          unsigned long long* __restrict__ pt_acc, DeviceCounters* __restrict__ dc,
                                                          int or_per_mcs) {
    allow_dependent_launch();
    grid_dependency_wait();                      // the pass that wrote the partial sums has completed
    if (dc) {                                    // CUDA-graph replay: this step's counters live on the device
        n_pt = dc->n_pt;
        series_row = dc->series_base ? dc->series_base + (size_t)dc->row * R * 5 : nullptr;
    }
    for (int k = threadIdx.x >> 5; k < R; k += 32)
        finalize_rank(partials, n_tiles, k, slot_at_rank[k], threadIdx.x & 31, obs_rank, obs_slot, series_row);
    __syncthreads();
    for (int pair = threadIdx.x; ; pair += blockDim.x) {
        const int k = (int)(n_pt & 1u) + 2 * pair;
        if (k + 1 >= R) break;
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
    if (dc) {
        __syncthreads();
        if (threadIdx.x == 0) { dc->n_met += 1u; dc->n_or += (uint32_t)or_per_mcs; dc->n_pt += 1u; dc->row += 1u; }
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

// The fast sin/cos, the fp64 window and the over-relaxation wrap are all stated for angles in [0, 2 pi]
// (R7): anything else entering through xy_set_state is reduced modulo 2 pi in double; in-range angles pass
// bit for bit; NaN / inf become 0.
__device__ __forceinline__ float angle_in_range(float t) {
    if (t >= 0.0f && t <= kTwoPiF) return t;
    if (!(fabsf(t) <= 3.0e38f)) return 0.0f;
    const double two_pi = 6.283185307179586476925;
    double r = fmod((double)t, two_pi);
    if (r < 0.0) r += two_pi;
    const float f = (float)r;
    return f > kTwoPiF ? kTwoPiF : f;
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
            float4 a = nat[0], b = nat[1];
            a.x = angle_in_range(a.x); a.y = angle_in_range(a.y); a.z = angle_in_range(a.z); a.w = angle_in_range(a.w);
            b.x = angle_in_range(b.x); b.y = angle_in_range(b.y); b.z = angle_in_range(b.z); b.w = angle_in_range(b.w);
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
__global__ void debug_sincos64_kernel(const double* x, double* c, double* s, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        double ss, cc; sincos_0_2pi(x[i], ss, cc); c[i] = cc; s[i] = ss;
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
