// lcs_kernels.cuh -- device code of liblcs_b200 (sm_100a).  See include/lcs.h for the contract and
// DESIGN.md section 6 for the kernel-by-kernel description.  Compiled with -fmad=false: a fused
// multiply-add happens only where fma() is written, so the push is bit-reproducible (DESIGN.md
// section 4, rules R1-R7).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace lcs {

constexpr int kBlock = 256;            // threads per tile CTA
constexpr int kIpt = 2;                // particles per thread = one 128-bit load per field
constexpr int kTile = kBlock * kIpt;   // particles per tile
constexpr int kWarps = kBlock / 32;
constexpr int kStay = 13;
constexpr int kNC = 27;                // destination codes

// Decoupled look-back descriptor word: [ epoch:30 | state:2 | value:32 ]
constexpr uint32_t kStAgg = 1u, kStPrefix = 2u;

struct Geom {
    int N, Px, Py, Pz, P, nx, ny, nz;
    int tiles_per_sub;                 // ceil(cap / kTile)
    int64_t cap, send_cap;
    double inv_dx, K_tau, L, L_below, gx, gy, gz;
};

struct Slabs {                         // SoA particle storage, P*cap slots each
    double* f[7];                      // x y z vx vy vz d
    int64_t* id;
    uint8_t* code;
};

struct Tables {
    uint32_t* count;                   // [P]    particles per slab
    uint32_t* cnt;                     // [P*32] per-(s,c) totals of the last step (27 used per row)
    uint32_t* recv_off;                // [P*32] slot in the receiver slab where segment (s,c) starts
    uint32_t* new_count;               // [P]
    uint64_t* desc;                    // [P*tiles_per_sub*32] look-back descriptors
    uint32_t* tile_excl;               // [P*tiles_per_sub*32] exclusive per-code prefix of each tile
    uint32_t* tile_cnt;                // [P*tiles_per_sub*32] per-code count of each tile
    unsigned int* ticket;              // tile ticket counter
    int* status;                       // sticky error word
    unsigned long long* n_migrated;    // migrants of the last migrate
    unsigned long long* n_total;
};

// ---------------------------------------------------------------------------------------------
// small helpers
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void raise(int* status, int code) { atomicCAS(status, 0, code); }

__device__ __forceinline__ uint64_t ld_relaxed_u64(const uint64_t* p)
{
    uint64_t v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed_u64(uint64_t* p, uint64_t v)
{
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// streaming (touched once) particle traffic: evict-first so it does not push the fluid bricks out of L2
__device__ __forceinline__ double2 ld_stream2(const double* p) { return __ldcs(reinterpret_cast<const double2*>(p)); }
__device__ __forceinline__ longlong2 ld_stream2(const int64_t* p) { return __ldcs(reinterpret_cast<const longlong2*>(p)); }
__device__ __forceinline__ void st_stream(double* p, double v) { __stcs(p, v); }
__device__ __forceinline__ void st_stream(int64_t* p, int64_t v) { __stcs(reinterpret_cast<long long*>(p), (long long)v); }

// exp(-z), z >= 0: range reduction by ln2 (hi/lo), degree-14 Taylor polynomial in Horner form with
// explicit fma, scaling by exponent arithmetic.  DESIGN.md R-3.
__device__ __forceinline__ double exp_neg(double z)
{
    if (!(z <= 708.0)) return (z != z) ? z : 0.0;
    const double y = -z;
    const double k = rint(y * 1.4426950408889634);
    double r = fma(-k, 6.93147180369123816490e-01, y);
    r = fma(-k, 1.90821492927058770002e-10, r);
    double p = 1.1470745597729725e-11;            // 1/14!
    p = fma(p, r, 1.6059043836821613e-10);        // 1/13!
    p = fma(p, r, 2.08767569878681e-09);          // 1/12!
    p = fma(p, r, 2.505210838544172e-08);         // 1/11!
    p = fma(p, r, 2.755731922398589e-07);         // 1/10!
    p = fma(p, r, 2.7557319223985893e-06);        // 1/9!
    p = fma(p, r, 2.48015873015873e-05);          // 1/8!
    p = fma(p, r, 0.0001984126984126984);         // 1/7!
    p = fma(p, r, 0.001388888888888889);          // 1/6!
    p = fma(p, r, 0.008333333333333333);          // 1/5!
    p = fma(p, r, 0.041666666666666664);          // 1/4!
    p = fma(p, r, 0.16666666666666666);           // 1/3!
    p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);
    p = fma(p, r, 1.0);
    // 2^k, k in [-1022, 0]: always a normal number, so the product is exact
    const long long bits = (long long)(1023 + (int)k) << 52;
    return p * __longlong_as_double(bits);
}

struct Axis { int i0, i1; double f; };

__device__ __forceinline__ Axis stencil_axis(double a, double inv_dx, int N)
{   // cell centre i sits at (i + 1/2) dx; periodic stencil (DESIGN R-9)
    Axis s;
    const double ga = fma(a, inv_dx, -0.5);
    const double fl = floor(ga);
    int i0 = (int)fl;
    s.f = ga - fl;
    i0 = max(-1, min(i0, N - 1));                 // memory safety for corrupt input only
    s.i0 = (i0 < 0) ? i0 + N : i0;
    s.i1 = (i0 + 1 >= N) ? i0 + 1 - N : i0 + 1;
    return s;
}

__device__ __forceinline__ double lerp(double p, double q, double f) { return fma(f, q - p, p); }

__device__ __forceinline__ double tri(const double* __restrict__ F, size_t r00, size_t r10, size_t r01,
                                      size_t r11, int i0, int i1, double fx, double fy, double fz)
{
    const double a0 = __ldg(F + r00 + i0), a1 = __ldg(F + r00 + i1);
    const double b0 = __ldg(F + r10 + i0), b1 = __ldg(F + r10 + i1);
    const double c0 = __ldg(F + r01 + i0), c1 = __ldg(F + r01 + i1);
    const double d0 = __ldg(F + r11 + i0), d1 = __ldg(F + r11 + i1);
    const double c00 = lerp(a0, a1, fx), c10 = lerp(b0, b1, fx);
    const double c01 = lerp(c0, c1, fx), c11 = lerp(d0, d1, fx);
    return lerp(lerp(c00, c10, fy), lerp(c01, c11, fy), fz);
}

struct Particle { double x, y, z, vx, vy, vz, d; };

// Per-block subdomain bounds in unwrapped cell index space.
struct SubBox { int lox, hix, loy, hiy, loz, hiz; };

// One axis of a2/a3: advance, wrap, classify.  Returns d in {-1,0,+1}; sets jump on violation.
__device__ __forceinline__ int advance_axis(double& a, double& v, double U, double g, double tau, double alpha,
                                            double b, double dt, const Geom& G, int lo, int hi, int n_a, bool& jump)
{
    const double vt = fma(tau, g, U);             // terminal velocity under frozen U
    const double w = v - vt;
    v = fma(w, alpha, vt);
    const double disp = fma(w, b, dt * vt);
    double xu = a + disp;
    int wrap = 0;
    if (xu < 0.0) { xu = xu + G.L; wrap = -1; if (xu >= G.L) xu = G.L_below; }
    else if (xu >= G.L) { xu = xu - G.L; wrap = 1; }
    a = xu;
    if (!(xu >= 0.0 && xu < G.L)) { jump = true; return 0; }
    int ic = (int)floor(xu * G.inv_dx);
    ic = max(0, min(ic, G.N - 1));
    const int icu = ic + wrap * G.N;              // unwrapped cell index (DESIGN R-14)
    const int dd = (icu >= hi) - (icu < lo);
    if (icu >= hi + n_a || icu < lo - n_a) jump = true;
    return dd;
}

// a1-a3 for one particle.  Returns the destination code.
__device__ __forceinline__ int push_particle(Particle& p, const double* __restrict__ u, const double* __restrict__ v,
                                             const double* __restrict__ w, const Geom& G, const SubBox& B, double dt,
                                             bool& jump)
{
    const Axis sx = stencil_axis(p.x, G.inv_dx, G.N);
    const Axis sy = stencil_axis(p.y, G.inv_dx, G.N);
    const Axis sz = stencil_axis(p.z, G.inv_dx, G.N);
    const size_t Ns = (size_t)G.N;
    const size_t r00 = Ns * (sy.i0 + Ns * sz.i0), r10 = Ns * (sy.i1 + Ns * sz.i0);
    const size_t r01 = Ns * (sy.i0 + Ns * sz.i1), r11 = Ns * (sy.i1 + Ns * sz.i1);
    const double Ux = tri(u, r00, r10, r01, r11, sx.i0, sx.i1, sx.f, sy.f, sz.f);
    const double Uy = tri(v, r00, r10, r01, r11, sx.i0, sx.i1, sx.f, sy.f, sz.f);
    const double Uz = tri(w, r00, r10, r01, r11, sx.i0, sx.i1, sx.f, sy.f, sz.f);
    const double tau = (G.K_tau * p.d) * p.d;     // tau_p = (rho_p/rho) d^2 / (18 nu)
    const double zz = dt / tau;
    const double alpha = exp_neg(zz);
    const double b = tau * (1.0 - alpha);
    const int dx = advance_axis(p.x, p.vx, Ux, G.gx, tau, alpha, b, dt, G, B.lox, B.hix, G.nx, jump);
    const int dy = advance_axis(p.y, p.vy, Uy, G.gy, tau, alpha, b, dt, G, B.loy, B.hiy, G.ny, jump);
    const int dz = advance_axis(p.z, p.vz, Uz, G.gz, tau, alpha, b, dt, G, B.loz, B.hiz, G.nz, jump);
    return (dx + 1) + 3 * (dy + 1) + 9 * (dz + 1);
}

__device__ __forceinline__ SubBox sub_box(const Geom& G, int s)
{
    const int px = s % G.Px, py = (s / G.Px) % G.Py, pz = s / (G.Px * G.Py);
    SubBox B;
    B.lox = px * G.nx; B.hix = B.lox + G.nx;
    B.loy = py * G.ny; B.hiy = B.loy + G.ny;
    B.loz = pz * G.nz; B.hiz = B.loz + G.nz;
    return B;
}

__device__ __forceinline__ int receiver_of(const Geom& G, int s, int c)
{
    const int px = s % G.Px, py = (s / G.Px) % G.Py, pz = s / (G.Px * G.Py);
    const int dx = c % 3 - 1, dy = (c / 3) % 3 - 1, dz = c / 9 - 1;
    const int qx = (px + dx + G.Px) % G.Px, qy = (py + dy + G.Py) % G.Py, qz = (pz + dz + G.Pz) % G.Pz;
    return qx + G.Px * (qy + G.Py * qz);
}

// ---------------------------------------------------------------------------------------------
// warp-level classification bookkeeping: six ballots per item row (x-,x+,y-,y+,z-,z+) + validity
// ---------------------------------------------------------------------------------------------
struct RowBallots { unsigned xm, xp, ym, yp, zm, zp, val; };

__device__ __forceinline__ RowBallots row_ballots(bool valid, int code)
{
    const int dx = code % 3, dy = (code / 3) % 3, dz = code / 9;   // 0,1,2 <-> -1,0,+1
    RowBallots r;
    r.val = __ballot_sync(0xffffffffu, valid);
    r.xm = __ballot_sync(0xffffffffu, valid && dx == 0);
    r.xp = __ballot_sync(0xffffffffu, valid && dx == 2);
    r.ym = __ballot_sync(0xffffffffu, valid && dy == 0);
    r.yp = __ballot_sync(0xffffffffu, valid && dy == 2);
    r.zm = __ballot_sync(0xffffffffu, valid && dz == 0);
    r.zp = __ballot_sync(0xffffffffu, valid && dz == 2);
    return r;
}

// lanes of the row whose particle has destination code c
__device__ __forceinline__ unsigned code_mask(const RowBallots& r, int c)
{
    const int dx = c % 3, dy = (c / 3) % 3, dz = c / 9;
    const unsigned mx = dx == 0 ? r.xm : (dx == 2 ? r.xp : r.val & ~(r.xm | r.xp));
    const unsigned my = dy == 0 ? r.ym : (dy == 2 ? r.yp : r.val & ~(r.ym | r.yp));
    const unsigned mz = dz == 0 ? r.zm : (dz == 2 ? r.zp : r.val & ~(r.zm | r.zp));
    return mx & my & mz;
}

// ---------------------------------------------------------------------------------------------
// K1: unfused push (a1-a4).  One CTA per (subdomain, tile); in place; codes + count table.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kBlock)
k_push(Geom G, Slabs S, Tables T, const double* __restrict__ fu, const double* __restrict__ fv,
       const double* __restrict__ fw, double dt)
{
    const int s = blockIdx.y;
    const int t = blockIdx.x;
    const uint32_t cnt_s = T.count[s];
    const int64_t first = (int64_t)t * kTile;
    if (first >= (int64_t)cnt_s) return;
    __shared__ uint32_t s_cnt[kNC];
    if (threadIdx.x < kNC) s_cnt[threadIdx.x] = 0;
    __syncthreads();
    const SubBox B = sub_box(G, s);
    const int64_t slot0 = first + 2 * (int64_t)threadIdx.x;      // even: 16-byte aligned
    const size_t base = (size_t)s * (size_t)G.cap + (size_t)slot0;
    const bool v0 = slot0 < (int64_t)cnt_s, v1 = slot0 + 1 < (int64_t)cnt_s;
    int c0 = kStay, c1 = kStay;
    bool jump = false;
    if (v0) {
        double2 q[7];
#pragma unroll
        for (int a = 0; a < 7; ++a) q[a] = ld_stream2(S.f[a] + base);
        Particle p0{q[0].x, q[1].x, q[2].x, q[3].x, q[4].x, q[5].x, q[6].x};
        Particle p1{q[0].y, q[1].y, q[2].y, q[3].y, q[4].y, q[5].y, q[6].y};
        c0 = push_particle(p0, fu, fv, fw, G, B, dt, jump);
        if (v1) c1 = push_particle(p1, fu, fv, fw, G, B, dt, jump);
        double2 o;
        o = make_double2(p0.x, p1.x);   __stcs(reinterpret_cast<double2*>(S.f[0] + base), o);
        o = make_double2(p0.y, p1.y);   __stcs(reinterpret_cast<double2*>(S.f[1] + base), o);
        o = make_double2(p0.z, p1.z);   __stcs(reinterpret_cast<double2*>(S.f[2] + base), o);
        o = make_double2(p0.vx, p1.vx); __stcs(reinterpret_cast<double2*>(S.f[3] + base), o);
        o = make_double2(p0.vy, p1.vy); __stcs(reinterpret_cast<double2*>(S.f[4] + base), o);
        o = make_double2(p0.vz, p1.vz); __stcs(reinterpret_cast<double2*>(S.f[5] + base), o);
        const uchar2 cc = make_uchar2((unsigned char)c0, (unsigned char)c1);
        *reinterpret_cast<uchar2*>(S.code + base) = cc;
    }
    if (jump) raise(T.status, -5);
    // a4: warp ballots -> per-code popc (lane c owns code c) -> shared -> one atomic per (tile, code)
    const RowBallots r0 = row_ballots(v0, c0), r1 = row_ballots(v1, c1);
    const int lane = threadIdx.x & 31;
    if (lane < kNC) {
        const uint32_t n = __popc(code_mask(r0, lane)) + __popc(code_mask(r1, lane));
        if (n) atomicAdd(&s_cnt[lane], n);
    }
    __syncthreads();
    if (threadIdx.x < kNC && s_cnt[threadIdx.x]) atomicAdd(&T.cnt[s * 32 + threadIdx.x], s_cnt[threadIdx.x]);
}

// ---------------------------------------------------------------------------------------------
// K2: tile pass of the migration (a5-a7), optionally with the push fused in front (a1-a4).
//   - per-code stable ranks by single-pass decoupled look-back over the tiles of one subdomain,
//     carried as a 27-vector (lane c of warp 0 owns code c);
//   - stayers written in place at their compacted slot;
//   - migrants written to the subdomain's send region, grouped by code inside the tile's chunk.
// Tiles take their index from an atomic ticket so every predecessor is resident or finished.
// `dep_zero` is always 0; it ties the id/field loads into the published aggregate so that a
// tile publishes only after its loads have completed (in-place compaction safety).
// ---------------------------------------------------------------------------------------------
template <bool kFused>
__global__ void __launch_bounds__(kBlock)
k_tile_pass(Geom G, Slabs S, Slabs Snd, Tables T, const double* __restrict__ fu, const double* __restrict__ fv,
            const double* __restrict__ fw, double dt, uint32_t epoch, unsigned long long dep_zero)
{
    __shared__ unsigned int s_ticket;
    __shared__ uint32_t s_wtot[kWarps][32];     // per-warp per-code counts, then exclusive prefix over warps
    __shared__ uint32_t s_excl[32];             // exclusive prefix of this tile (over earlier tiles of s)
    __shared__ uint32_t s_codeoff[32];          // offset of code c inside this tile's send chunk
    __shared__ int64_t s_sendbase;              // first send slot of this tile's chunk, -1 = overflow

    if (threadIdx.x == 0) s_ticket = atomicAdd(T.ticket, 1u);
    __syncthreads();
    const unsigned int g = s_ticket;
    const int s = g / G.tiles_per_sub;
    const int t = g % G.tiles_per_sub;
    const uint32_t cnt_s = T.count[s];
    const int64_t first = (int64_t)t * kTile;
    if (first >= (int64_t)cnt_s) return;
    const bool last_tile = first + kTile >= (int64_t)cnt_s;

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t slot0 = first + 2 * (int64_t)threadIdx.x;
    const size_t slab0 = (size_t)s * (size_t)G.cap;
    const size_t base = slab0 + (size_t)slot0;
    const bool v0 = slot0 < (int64_t)cnt_s, v1 = slot0 + 1 < (int64_t)cnt_s;

    Particle p0, p1;
    int64_t id0 = 0, id1 = 0;
    int c0 = kStay, c1 = kStay;
    bool jump = false;
    unsigned long long dep = 0;
    if (v0) {
        double2 q[7];
#pragma unroll
        for (int a = 0; a < 7; ++a) q[a] = ld_stream2(S.f[a] + base);
        const longlong2 qi = ld_stream2(S.id + base);
        p0 = Particle{q[0].x, q[1].x, q[2].x, q[3].x, q[4].x, q[5].x, q[6].x};
        p1 = Particle{q[0].y, q[1].y, q[2].y, q[3].y, q[4].y, q[5].y, q[6].y};
        id0 = qi.x; id1 = qi.y;
        if (kFused) {
            const SubBox B = sub_box(G, s);
            c0 = push_particle(p0, fu, fv, fw, G, B, dt, jump);
            if (v1) c1 = push_particle(p1, fu, fv, fw, G, B, dt, jump);
            dep = (unsigned long long)(id0 ^ id1);
        } else {
            const uchar2 cc = *reinterpret_cast<const uchar2*>(S.code + base);
            c0 = min((int)cc.x, 26);
            c1 = v1 ? min((int)cc.y, 26) : kStay;
            dep = (unsigned long long)(id0 ^ id1);
#pragma unroll
            for (int a = 0; a < 7; ++a)
                dep ^= (unsigned long long)(__double_as_longlong(q[a].x) ^ __double_as_longlong(q[a].y));
        }
        dep &= dep_zero;                          // == 0, but only known at run time
    }
    if (jump) raise(T.status, -5);

    // --- in-warp ranks and per-warp totals --------------------------------------------------
    const RowBallots r0 = row_ballots(v0 || dep != 0, c0), r1 = row_ballots(v1, c1);
    const unsigned lt = (1u << lane) - 1u;
    const uint32_t rank0 = __popc(code_mask(r0, c0) & lt) + __popc(code_mask(r1, c0) & lt);
    const uint32_t rank1 = __popc(code_mask(r0, c1) & lt) + __popc(code_mask(r1, c1) & lt) + ((v0 && c0 == c1) ? 1u : 0u);
    s_wtot[warp][lane] = (lane < kNC) ? (uint32_t)(__popc(code_mask(r0, lane)) + __popc(code_mask(r1, lane))) : 0u;
    __syncthreads();

    // --- warp 0: block aggregate, publish, look back ------------------------------------------
    if (warp == 0) {
        uint32_t agg = 0;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) { const uint32_t v = s_wtot[w][lane]; s_wtot[w][lane] = agg; agg += v; }
        uint64_t* my_desc = T.desc + ((size_t)s * G.tiles_per_sub + t) * 32;
        const uint64_t tag = (uint64_t)(epoch << 2) << 32;
        uint32_t excl = 0;
        if (t == 0) {
            st_relaxed_u64(my_desc + lane, tag | ((uint64_t)kStPrefix << 32) | agg);
        } else {
            st_relaxed_u64(my_desc + lane, tag | ((uint64_t)kStAgg << 32) | agg);
            int j = t - 1;
            while (true) {
                const uint64_t* pd = T.desc + ((size_t)s * G.tiles_per_sub + j) * 32 + lane;
                uint64_t wv = ld_relaxed_u64(pd);
                while ((uint32_t)(wv >> 34) != epoch || ((uint32_t)(wv >> 32) & 3u) == 0u) { __nanosleep(20); wv = ld_relaxed_u64(pd); }
                excl += (uint32_t)wv;
                if (((uint32_t)(wv >> 32) & 3u) == kStPrefix) break;
                --j;
            }
            st_relaxed_u64(my_desc + lane, tag | ((uint64_t)kStPrefix << 32) | (uint64_t)(excl + agg));
        }
        s_excl[lane] = excl;
        const size_t trow = ((size_t)s * G.tiles_per_sub + t) * 32 + lane;
        T.tile_excl[trow] = excl;
        T.tile_cnt[trow] = agg;
        if (last_tile) T.cnt[s * 32 + lane] = excl + agg;      // a4/a5 totals of subdomain s
        // offsets of each code's run inside this tile's send chunk, and the chunk's position
        const uint32_t magg = (lane < kNC && lane != kStay) ? agg : 0u;
        const uint32_t mexc = (lane < kNC && lane != kStay) ? excl : 0u;
        uint32_t inc = magg, tot_excl = mexc;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t nb = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += nb;
            tot_excl += __shfl_xor_sync(0xffffffffu, tot_excl, o);
        }
        s_codeoff[lane] = inc - magg;
        const uint32_t n_mig_tile = __shfl_sync(0xffffffffu, inc, 31);
        if (lane == 0) {
            int64_t sb = (int64_t)s * G.send_cap + (int64_t)tot_excl;
            if ((int64_t)tot_excl + (int64_t)n_mig_tile > G.send_cap) { raise(T.status, -4); sb = -1; }
            s_sendbase = sb;
        }
    }
    __syncthreads();

    // --- scatter: stayers compact in place, migrants to the send chunk ---------------------------
    const int64_t sendbase = s_sendbase;
#pragma unroll
    for (int e = 0; e < kIpt; ++e) {
        const bool valid = e == 0 ? v0 : v1;
        if (!valid) continue;
        const int c = e == 0 ? c0 : c1;
        const Particle& p = e == 0 ? p0 : p1;
        const int64_t pid = e == 0 ? id0 : id1;
        const uint32_t in_tile = s_wtot[warp][c] + (e == 0 ? rank0 : rank1);
        const bool stay = c == kStay;
        if (!stay && sendbase < 0) continue;
        const size_t dst = stay ? slab0 + (size_t)s_excl[kStay] + in_tile
                                : (size_t)sendbase + s_codeoff[c] + in_tile;
        st_stream((stay ? S.f[0] : Snd.f[0]) + dst, p.x);
        st_stream((stay ? S.f[1] : Snd.f[1]) + dst, p.y);
        st_stream((stay ? S.f[2] : Snd.f[2]) + dst, p.z);
        st_stream((stay ? S.f[3] : Snd.f[3]) + dst, p.vx);
        st_stream((stay ? S.f[4] : Snd.f[4]) + dst, p.vy);
        st_stream((stay ? S.f[5] : Snd.f[5]) + dst, p.vz);
        st_stream((stay ? S.f[6] : Snd.f[6]) + dst, p.d);
        st_stream((stay ? S.id : Snd.id) + dst, pid);
    }
}

// ---------------------------------------------------------------------------------------------
// K3: table scan (a5 at table level).  stay[s], receive offsets in the fixed order (s ascending,
// c ascending), new counts, overflow flag, totals.  One CTA, thread r owns receiver r.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_table(Geom G, Tables T)
{
    __shared__ unsigned long long s_mig, s_tot;
    if (threadIdx.x == 0) { s_mig = 0; s_tot = 0; *T.ticket = 0u; }
    __syncthreads();
    unsigned long long my_mig = 0, my_tot = 0;
    for (int r = threadIdx.x; r < G.P; r += blockDim.x) {
        // the 26 incoming segments (s_c, c): s_c is the neighbour of r in direction -d(c)
        int src[kNC];
        uint32_t len[kNC];
        const int rx = r % G.Px, ry = (r / G.Px) % G.Py, rz = r / (G.Px * G.Py);
        for (int c = 0; c < kNC; ++c) {
            const int dx = c % 3 - 1, dy = (c / 3) % 3 - 1, dz = c / 9 - 1;
            const int sx = (rx - dx + G.Px) % G.Px, sy = (ry - dy + G.Py) % G.Py, sz = (rz - dz + G.Pz) % G.Pz;
            const int sc = sx + G.Px * (sy + G.Py * sz);
            src[c] = sc;
            len[c] = (T.count[sc] == 0) ? 0u : T.cnt[sc * 32 + c];
        }
        const uint32_t stay = (T.count[r] == 0) ? 0u : T.cnt[r * 32 + kStay];
        // fixed order: s ascending, then c ascending (DESIGN R-12).  Rank of (src[c], c) among the 26.
        unsigned long long fill = stay;
        uint32_t off[kNC];
        for (int c = 0; c < kNC; ++c) {
            if (c == kStay) { off[c] = 0; continue; }
            unsigned long long before = stay;
            for (int c2 = 0; c2 < kNC; ++c2) {
                if (c2 == kStay) continue;
                if (src[c2] < src[c] || (src[c2] == src[c] && c2 < c)) before += len[c2];
            }
            off[c] = (uint32_t)min(before, (unsigned long long)0xffffffffu);
            fill += len[c];
            my_mig += len[c];
        }
        if (fill > (unsigned long long)G.cap) { raise(T.status, -4); fill = (unsigned long long)G.cap; }
        for (int c = 0; c < kNC; ++c)
            if (c != kStay) T.recv_off[src[c] * 32 + c] = off[c];
        T.new_count[r] = (uint32_t)fill;
        my_tot += fill;
    }
    atomicAdd(&s_mig, my_mig);
    atomicAdd(&s_tot, my_tot);
    __syncthreads();
    if (threadIdx.x == 0) { *T.n_migrated = s_mig; *T.n_total = s_tot; }
}

// ---------------------------------------------------------------------------------------------
// K4: unpack / append (a8).  One CTA per tile chunk of the send pool; copies each code's run to
// slab[receiver(s,c)] + recv_off[s][c] + (exclusive per-code prefix of the tile).
// ---------------------------------------------------------------------------------------------
constexpr int kUnpackBlock = 64;

__global__ void __launch_bounds__(kUnpackBlock)
k_unpack(Geom G, Slabs S, Slabs Snd, Tables T)
{
    const int s = blockIdx.y, t = blockIdx.x;
    const uint32_t cnt_s = T.count[s];
    if ((int64_t)t * kTile >= (int64_t)cnt_s) return;
    if (*T.status != 0) return;                                 // contents unspecified after an error
    __shared__ uint32_t s_off[32];       // start of code c inside the chunk
    __shared__ uint32_t s_len[32];       // length of code c's run
    __shared__ int64_t s_dst[32];        // destination slot of the first element of code c's run
    __shared__ uint32_t s_n;
    __shared__ int64_t s_src;
    const int lane = threadIdx.x;
    if (lane < 32) {
        const size_t trow = ((size_t)s * G.tiles_per_sub + t) * 32 + lane;
        const bool mig = lane < kNC && lane != kStay;
        const uint32_t agg = mig ? T.tile_cnt[trow] : 0u;
        const uint32_t exc = mig ? T.tile_excl[trow] : 0u;
        uint32_t inc = agg, tot_excl = exc;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t nb = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += nb;
            tot_excl += __shfl_xor_sync(0xffffffffu, tot_excl, o);
        }
        s_off[lane] = inc - agg;
        s_len[lane] = agg;
        int64_t d = -1;
        if (mig) {
            const int r = receiver_of(G, s, lane);
            d = (int64_t)r * G.cap + (int64_t)T.recv_off[s * 32 + lane] + (int64_t)exc;
            // memory safety if counts were clamped after an overflow
            if ((int64_t)T.recv_off[s * 32 + lane] + (int64_t)exc + (int64_t)agg > G.cap) d = -1;
        }
        s_dst[lane] = d;
        if (lane == 31) s_n = inc;
        if (lane == 0) s_src = (int64_t)s * G.send_cap + (int64_t)tot_excl;
    }
    __syncthreads();
    const uint32_t n = s_n;
    const int64_t src0 = s_src;
    for (uint32_t i = threadIdx.x; i < n; i += kUnpackBlock) {
        int c = 0;
#pragma unroll 1
        for (int k = 1; k < kNC; ++k) c = (s_len[k] != 0u && s_off[k] <= i) ? k : c;   // last non-empty run starting at or before i
        if (s_dst[c] < 0) continue;
        const size_t dst = (size_t)(s_dst[c] + (int64_t)(i - s_off[c]));
        const size_t src = (size_t)(src0 + (int64_t)i);
#pragma unroll
        for (int a = 0; a < 7; ++a) S.f[a][dst] = __ldcs(Snd.f[a] + src);
        S.id[dst] = __ldcs(reinterpret_cast<const long long*>(Snd.id) + src);
    }
}

// counts <- new counts (after unpack)
__global__ void k_commit_counts(Geom G, Tables T)
{
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r < G.P && *T.status == 0) T.count[r] = T.new_count[r];
}

// ---------------------------------------------------------------------------------------------
// accessors
// ---------------------------------------------------------------------------------------------
__global__ void k_counts_out(Geom G, Tables T, int64_t* out, int64_t* prefix)
{   // one CTA; out[P] (may be null) and exclusive prefix[P+1] (may be null)
    __shared__ int64_t s_run;
    __shared__ int64_t sh[256];
    if (threadIdx.x == 0) s_run = 0;
    __syncthreads();
    for (int b = 0; b < G.P; b += blockDim.x) {
        const int r = b + threadIdx.x;
        const int64_t v = r < G.P ? (int64_t)T.count[r] : 0;
        // block inclusive scan (simple Hillis-Steele through shared memory)
        sh[threadIdx.x] = v;
        __syncthreads();
        for (int o = 1; o < (int)blockDim.x; o <<= 1) {
            const int64_t add = threadIdx.x >= (unsigned)o ? sh[threadIdx.x - o] : 0;
            __syncthreads();
            sh[threadIdx.x] += add;
            __syncthreads();
        }
        const int64_t incl = sh[threadIdx.x] + s_run;
        if (r < G.P) {
            if (out) out[r] = v;
            if (prefix) prefix[r] = incl - v;
        }
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) s_run = incl;
        __syncthreads();
    }
    if (threadIdx.x == 0 && prefix) prefix[G.P] = s_run;
}

struct OutPtrs { double* f[7]; int64_t* id; uint8_t* code; };

__global__ void __launch_bounds__(kBlock)
k_copy_out(Geom G, Slabs S, Tables T, const int64_t* __restrict__ prefix, OutPtrs O, int codes_valid)
{
    const int s = blockIdx.y, t = blockIdx.x;
    const int64_t cnt_s = (int64_t)T.count[s];
    const int64_t first = (int64_t)t * kTile;
    if (first >= cnt_s) return;
    const int64_t obase = prefix[s];
    const size_t slab0 = (size_t)s * (size_t)G.cap;
    for (int64_t i = first + threadIdx.x; i < min(first + kTile, cnt_s); i += kBlock) {
#pragma unroll
        for (int a = 0; a < 7; ++a) if (O.f[a]) O.f[a][obase + i] = S.f[a][slab0 + i];
        if (O.id) O.id[obase + i] = S.id[slab0 + i];
        if (O.code) O.code[obase + i] = codes_valid ? S.code[slab0 + i] : (uint8_t)kStay;
    }
}

__global__ void k_table_out(Geom G, Tables T, int64_t* out, int pushed)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= G.P * kNC) return;
    const int s = i / kNC, c = i % kNC;
    int64_t v;
    if (pushed) v = T.count[s] ? (int64_t)T.cnt[s * 32 + c] : 0;
    else v = (c == kStay) ? (int64_t)T.count[s] : 0;
    out[i] = v;
}

// ---------------------------------------------------------------------------------------------
// lcs_set_particles: stable binning by owner (counting sort with P buckets), three kernels
// ---------------------------------------------------------------------------------------------
constexpr int kSetTile = 4096;

__device__ __forceinline__ int cell_clamped(double a, double inv_dx, int N)
{
    int i = (int)floor(a * inv_dx);
    return max(0, min(i, N - 1));
}

__global__ void __launch_bounds__(256)
k_set_owner(Geom G, Tables T, int64_t n, const double* __restrict__ x, const double* __restrict__ y,
            const double* __restrict__ z, int32_t* __restrict__ owner, uint32_t* __restrict__ tilehist)
{
    extern __shared__ uint32_t s_hist[];
    for (int p = threadIdx.x; p < G.P; p += blockDim.x) s_hist[p] = 0;
    __syncthreads();
    const int64_t first = (int64_t)blockIdx.x * kSetTile;
    bool bad = false;
    for (int64_t i = first + threadIdx.x; i < min(first + kSetTile, n); i += blockDim.x) {
        const double px = x[i], py = y[i], pz = z[i];
        if (!(px >= 0.0 && px < G.L && py >= 0.0 && py < G.L && pz >= 0.0 && pz < G.L)) bad = true;
        const int ow = cell_clamped(px, G.inv_dx, G.N) / G.nx
                     + G.Px * (cell_clamped(py, G.inv_dx, G.N) / G.ny + G.Py * (cell_clamped(pz, G.inv_dx, G.N) / G.nz));
        owner[i] = ow;
        atomicAdd(&s_hist[ow], 1u);
    }
    if (bad) raise(T.status, -6);
    __syncthreads();
    for (int p = threadIdx.x; p < G.P; p += blockDim.x) tilehist[(size_t)blockIdx.x * G.P + p] = s_hist[p];
}

__global__ void k_set_scan(Geom G, Tables T, int ntiles, uint32_t* __restrict__ tilehist, int64_t n)
{   // thread p: exclusive scan of bucket p over tiles (in place), total -> count[p]
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p == 0) *T.n_total = (unsigned long long)n;
    if (p >= G.P) return;
    uint64_t run = 0;
    for (int t = 0; t < ntiles; ++t) {
        const uint32_t v = tilehist[(size_t)t * G.P + p];
        tilehist[(size_t)t * G.P + p] = (uint32_t)min(run, (uint64_t)0xffffffffu);
        run += v;
    }
    if (run > (uint64_t)G.cap) { raise(T.status, -4); run = (uint64_t)G.cap; }
    T.count[p] = (uint32_t)run;
    for (int c = 0; c < 32; ++c) T.cnt[p * 32 + c] = (c == kStay) ? (uint32_t)run : 0u;
}

struct InPtrs { const double* f[7]; const int64_t* id; };

__global__ void __launch_bounds__(128)
k_set_scatter(Geom G, Slabs S, int64_t n, InPtrs I, const int32_t* __restrict__ owner,
              const uint32_t* __restrict__ tileoff, int warps_per_block)
{   // one warp per tile, sequential 32-particle rounds: stable rank = running bucket counter + match rank
    extern __shared__ uint32_t s_run[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t tile = (int64_t)blockIdx.x * warps_per_block + warp;
    const int64_t first = tile * kSetTile;
    if (first >= n) return;
    uint32_t* run = s_run + (size_t)warp * G.P;
    for (int p = lane; p < G.P; p += 32) run[p] = tileoff[(size_t)tile * G.P + p];
    __syncwarp();
    const int64_t end = min(first + kSetTile, n);
    for (int64_t i0 = first; i0 < end; i0 += 32) {
        const int64_t i = i0 + lane;
        const bool valid = i < end;
        const int ow = valid ? owner[i] : -1 - lane;            // distinct dummies never match
        const unsigned m = __match_any_sync(0xffffffffu, ow);
        const uint32_t rank = __popc(m & ((1u << lane) - 1u));
        uint32_t slot = 0;
        if (valid) slot = run[ow] + rank;
        __syncwarp();
        if (valid && rank == (uint32_t)__popc(m) - 1u) run[ow] = slot + 1u;   // last lane of the group
        __syncwarp();
        if (valid && (int64_t)slot < G.cap) {
            const size_t dst = (size_t)ow * (size_t)G.cap + slot;
#pragma unroll
            for (int a = 0; a < 7; ++a) S.f[a][dst] = I.f[a][i];
            S.id[dst] = I.id[i];
        }
    }
}

}  // namespace lcs
