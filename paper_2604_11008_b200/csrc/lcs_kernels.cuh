// lcs_kernels.cuh -- device code of liblcs_b200 (sm_100a).  See include/lcs.h for the contract and
// DESIGN.md section 6 for the kernel-by-kernel description.  Compiled with -fmad=false: a fused
// multiply-add happens only where fma() is written, so the push is bit-reproducible (DESIGN.md
// section 4, rules R1-R7).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace lcs {

#ifndef LCS_BLOCK
#define LCS_BLOCK 256
#endif
#ifndef LCS_MIN_BLOCKS
#define LCS_MIN_BLOCKS 2
#endif
constexpr int kBlock = LCS_BLOCK;      // threads per tile CTA
constexpr int kMinBlocks = LCS_MIN_BLOCKS;   // CTAs per SM the tile pass is compiled for
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
    uint64_t* desc;                    // [P*tiles_per_sub*2] look-back descriptors: (stay, migrant) words
    uint32_t* tile_start;              // [P+1] compact prefix of non-empty tiles per subdomain
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

// Fluid is held as one 32-byte record per cell: (u, v, w, 0) -- one L2 sector and one 256-bit load per
// stencil corner instead of three scattered 8-byte loads.
struct alignas(32) Cell { double u, v, w, pad; };

__device__ __forceinline__ Cell ld_cell(const double* __restrict__ F4, size_t cell)
{
    Cell r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f64 {%0,%1,%2,%3}, [%4];"
                 : "=d"(r.u), "=d"(r.v), "=d"(r.w), "=d"(r.pad) : "l"(F4 + 4 * cell));
    return r;
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
__device__ __forceinline__ int push_particle(Particle& p, const double* __restrict__ F4, const Geom& G,
                                             const SubBox& B, double dt, bool& jump)
{
    const Axis sx = stencil_axis(p.x, G.inv_dx, G.N);
    const Axis sy = stencil_axis(p.y, G.inv_dx, G.N);
    const Axis sz = stencil_axis(p.z, G.inv_dx, G.N);
    const size_t Ns = (size_t)G.N;
    const size_t r00 = Ns * (sy.i0 + Ns * sz.i0), r10 = Ns * (sy.i1 + Ns * sz.i0);
    const size_t r01 = Ns * (sy.i0 + Ns * sz.i1), r11 = Ns * (sy.i1 + Ns * sz.i1);
    double Ux, Uy, Uz;
    {
        const Cell a0 = ld_cell(F4, r00 + sx.i0), a1 = ld_cell(F4, r00 + sx.i1);
        const Cell b0 = ld_cell(F4, r10 + sx.i0), b1 = ld_cell(F4, r10 + sx.i1);
        const Cell c0 = ld_cell(F4, r01 + sx.i0), c1 = ld_cell(F4, r01 + sx.i1);
        const Cell d0 = ld_cell(F4, r11 + sx.i0), d1 = ld_cell(F4, r11 + sx.i1);
        // same lerp order as the definition: x, then y, then z
        Ux = lerp(lerp(lerp(a0.u, a1.u, sx.f), lerp(b0.u, b1.u, sx.f), sy.f),
                  lerp(lerp(c0.u, c1.u, sx.f), lerp(d0.u, d1.u, sx.f), sy.f), sz.f);
        Uy = lerp(lerp(lerp(a0.v, a1.v, sx.f), lerp(b0.v, b1.v, sx.f), sy.f),
                  lerp(lerp(c0.v, c1.v, sx.f), lerp(d0.v, d1.v, sx.f), sy.f), sz.f);
        Uz = lerp(lerp(lerp(a0.w, a1.w, sx.f), lerp(b0.w, b1.w, sx.f), sy.f),
                  lerp(lerp(c0.w, c1.w, sx.f), lerp(d0.w, d1.w, sx.f), sy.f), sz.f);
    }
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
// K0: lcs_set_fluid -- repack the three x-fastest arrays into one (u,v,w,0) record per cell
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_repack_fluid(size_t ncell, const double* __restrict__ u, const double* __restrict__ v, const double* __restrict__ w,
               double* __restrict__ F4)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < ncell; i += (size_t)gridDim.x * blockDim.x) {
        const double4 r = make_double4(__ldcs(u + i), __ldcs(v + i), __ldcs(w + i), 0.0);
        *reinterpret_cast<double4*>(F4 + 4 * i) = r;
    }
}

// ---------------------------------------------------------------------------------------------
// K1: unfused push (a1-a4).  One CTA per (subdomain, tile); in place; codes + count table.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kBlock)
k_push(Geom G, Slabs S, Tables T, const double* __restrict__ F4, double dt)
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
        c0 = push_particle(p0, F4, G, B, dt, jump);
        if (v1) c1 = push_particle(p1, F4, G, B, dt, jump);
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
//   Persistent CTAs; each takes tiles from an atomic ticket (so every predecessor of a tile is
//   resident or finished) and maps the ticket to (subdomain, tile) through the compact prefix
//   tile_start[] (empty tiles never get a ticket).  Per tile:
//   - in-tile per-code stable ranks from warp ballots (lane c owns code c);
//   - single-pass decoupled look-back over the tiles of the SAME subdomain with a 32-wide window
//     (lane L inspects predecessor t-1-L), carrying two running sums: stayers and migrants;
//   - stayers written in place at their compacted slot; migrants written to the subdomain's send
//     region at (migrant prefix) + (offset of their code's run in the tile chunk) + (in-tile rank).
//   The per-code cross-tile prefix needed by the unpack is produced afterwards by k_code_scan
//   from tile_cnt[] (it is not on the critical path of the look-back).
// `dep_zero` is always 0; it ties the id/field loads into the published aggregate so that a
// tile publishes only after its loads have completed (in-place compaction safety).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t warp_sum(uint32_t v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// one window step of the look-back for one of the two running sums; returns true when a PREFIX was found
__device__ __forceinline__ bool window_step(uint64_t w, bool beyond_start, int lane, uint32_t& excl)
{
    const bool is_prefix = beyond_start || ((uint32_t)(w >> 32) & 3u) == kStPrefix;
    const unsigned pm = __ballot_sync(0xffffffffu, is_prefix);
    const int first = pm ? (__ffs(pm) - 1) : 32;               // nearest predecessor holding a prefix
    const uint32_t v = (lane <= first && !beyond_start) ? (uint32_t)w : 0u;
    excl += warp_sum(v);
    return pm != 0u;
}

// A pushed tile staged in shared memory in OUTPUT order: stayers first (stable), then the migrants
// grouped by destination code (stable inside each code).
struct TileBuf {
    double f[7][kTile];
    long long id[kTile];
};

struct TileCtl {
    uint32_t wtot[kWarps][32];      // per-warp per-code counts of the tile being pushed
    uint32_t stay_excl;             // look-back result of the tile being resolved
    long long sendbase;             // first send slot of its chunk, -1 = send region overflow
    unsigned int next_ticket;
};

// Per-tile facts carried from its push to its resolve one iteration later (all CTA-uniform).
struct TileInfo { int s, t; uint32_t n_stay, n_mig, cnt_s; bool valid; };

template <bool kFused>
__global__ void __launch_bounds__(kBlock, kMinBlocks)
k_tile_pass(Geom G, Slabs S, Slabs Snd, Tables T, const double* __restrict__ F4, double dt, uint32_t epoch,
            unsigned long long dep_zero)
{
    extern __shared__ __align__(16) unsigned char s_raw[];
    TileBuf* buf = reinterpret_cast<TileBuf*>(s_raw);                                   // [2]
    uint32_t* s_tile_start = reinterpret_cast<uint32_t*>(s_raw + 2 * sizeof(TileBuf));  // [P+1]
    __shared__ TileCtl sm;

    for (int i = threadIdx.x; i <= G.P; i += kBlock) s_tile_start[i] = T.tile_start[i];
    if (threadIdx.x == 0) sm.next_ticket = atomicAdd(T.ticket, 1u);
    __syncthreads();
    const unsigned int n_active = s_tile_start[G.P];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint64_t tag = (uint64_t)(epoch << 2) << 32;

    TileInfo prev; prev.valid = false; prev.s = prev.t = 0; prev.n_stay = prev.n_mig = prev.cnt_s = 0;
    for (int it = 0;; ++it) {
        const int b = it & 1;
        const unsigned int g = sm.next_ticket;
        TileInfo cur; cur.valid = g < n_active; cur.s = cur.t = 0; cur.n_stay = cur.n_mig = cur.cnt_s = 0;
        if (!cur.valid && !prev.valid) break;

        // ============ push phase of tile g: load, (push,) rank, stage into buf[b], publish aggregate ============
        if (cur.valid) {
            int lo = 0, hi = G.P;                                       // largest s with tile_start[s] <= g
            while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (s_tile_start[mid] <= g) lo = mid; else hi = mid; }
            cur.s = lo;
            cur.t = (int)(g - s_tile_start[lo]);
            cur.cnt_s = T.count[lo];
            const int64_t first = (int64_t)cur.t * kTile;
            const int64_t slot0 = first + 2 * (int64_t)threadIdx.x;
            const size_t base = (size_t)cur.s * (size_t)G.cap + (size_t)slot0;
            const bool v0 = slot0 < (int64_t)cur.cnt_s, v1 = slot0 + 1 < (int64_t)cur.cnt_s;

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
                    const SubBox B = sub_box(G, cur.s);
                    c0 = push_particle(p0, F4, G, B, dt, jump);
                    if (v1) c1 = push_particle(p1, F4, G, B, dt, jump);
                } else {
                    const uchar2 cc = *reinterpret_cast<const uchar2*>(S.code + base);
                    c0 = min((int)cc.x, 26);
                    c1 = v1 ? min((int)cc.y, 26) : kStay;
                }
            }
            if (jump) raise(T.status, -5);

            // in-warp ranks and per-warp totals
            const RowBallots r0 = row_ballots(v0, c0), r1 = row_ballots(v1, c1);
            const unsigned lt = (1u << lane) - 1u;
            const uint32_t rank0 = __popc(code_mask(r0, c0) & lt) + __popc(code_mask(r1, c0) & lt);
            const uint32_t rank1 = __popc(code_mask(r0, c1) & lt) + __popc(code_mask(r1, c1) & lt) + ((v0 && c0 == c1) ? 1u : 0u);
            sm.wtot[warp][lane] = (lane < kNC) ? (uint32_t)(__popc(code_mask(r0, lane)) + __popc(code_mask(r1, lane))) : 0u;
            __syncthreads();                                                                             // B1
            // every warp: lane c sums code c over the warps -> its own exclusive prefix and the tile total
            uint32_t wexcl = 0, agg = 0;
#pragma unroll
            for (int w = 0; w < kWarps; ++w) { const uint32_t v = sm.wtot[w][lane]; if (w < warp) wexcl += v; agg += v; }
            const uint32_t magg = (lane < kNC && lane != kStay) ? agg : 0u;
            uint32_t inc = magg;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t nb = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += nb;
            }
            cur.n_mig = __shfl_sync(0xffffffffu, inc, 31);
            cur.n_stay = __shfl_sync(0xffffffffu, agg, kStay);
            // position of code c's run in the staged tile: stayers at 0, migrants after them in code order
            const uint32_t run_start = (lane == kStay) ? 0u : cur.n_stay + (inc - magg);
            const uint32_t my_base = run_start + wexcl;            // lane c: first staged slot of this warp's code-c particles
            TileBuf& B = buf[b];
            if (v0) {
                const uint32_t pos = __shfl_sync(0xffffffffu, my_base, c0) + rank0;
                B.f[0][pos] = p0.x; B.f[1][pos] = p0.y; B.f[2][pos] = p0.z; B.f[3][pos] = p0.vx;
                B.f[4][pos] = p0.vy; B.f[5][pos] = p0.vz; B.f[6][pos] = p0.d; B.id[pos] = id0;
            } else (void)__shfl_sync(0xffffffffu, my_base, 0);
            if (v1) {
                const uint32_t pos = __shfl_sync(0xffffffffu, my_base, c1) + rank1;
                B.f[0][pos] = p1.x; B.f[1][pos] = p1.y; B.f[2][pos] = p1.z; B.f[3][pos] = p1.vx;
                B.f[4][pos] = p1.vy; B.f[5][pos] = p1.vz; B.f[6][pos] = p1.d; B.id[pos] = id1;
            } else (void)__shfl_sync(0xffffffffu, my_base, 0);
            if (warp == 0) {
                // The staged copies above are this warp's own; the other warps' loads are ordered before the
                // publish by barrier B1 (their ballots consumed the loaded values) -- see DESIGN.md 6.3.
                const size_t tile_row = (size_t)cur.s * G.tiles_per_sub + cur.t;
                T.tile_cnt[tile_row * 32 + lane] = agg;
                if (lane < 2) {
                    const uint32_t mine = lane == 0 ? cur.n_stay : cur.n_mig;
                    const uint32_t st = cur.t == 0 ? kStPrefix : kStAgg;
                    st_relaxed_u64(T.desc + tile_row * 2 + lane, tag | ((uint64_t)st << 32) | mine);
                }
            }
        }

        // ============ resolve phase of the previous tile: windowed look-back (warp 0) ============
        if (prev.valid && warp == 0) {
            uint32_t excl_stay = 0, excl_mig = 0;
            if (prev.t > 0) {
                bool done_s = false, done_m = false;
                for (int nearest = prev.t - 1; !(done_s && done_m); nearest -= 32) {
                    const int j = nearest - lane;
                    const bool beyond = j < 0;                       // before the subdomain's first tile: prefix 0
                    uint64_t wa = 0, wb = 0;
                    if (!beyond) {
                        const uint64_t* pd = T.desc + ((size_t)prev.s * G.tiles_per_sub + j) * 2;
                        wa = ld_relaxed_u64(pd);
                        wb = ld_relaxed_u64(pd + 1);
                        while ((uint32_t)(wa >> 34) != epoch || ((uint32_t)(wa >> 32) & 3u) == 0u ||
                               (uint32_t)(wb >> 34) != epoch || ((uint32_t)(wb >> 32) & 3u) == 0u) {
                            __nanosleep(20);
                            wa = ld_relaxed_u64(pd);
                            wb = ld_relaxed_u64(pd + 1);
                        }
                    }
                    if (!done_s) done_s = window_step(wa, beyond, lane, excl_stay);
                    if (!done_m) done_m = window_step(wb, beyond, lane, excl_mig);
                }
                if (lane < 2) {
                    const uint32_t incl = lane == 0 ? excl_stay + prev.n_stay : excl_mig + prev.n_mig;
                    st_relaxed_u64(T.desc + ((size_t)prev.s * G.tiles_per_sub + prev.t) * 2 + lane,
                                   tag | ((uint64_t)kStPrefix << 32) | (uint64_t)incl);
                }
            }
            if (lane == 0) {
                sm.stay_excl = excl_stay;
                long long sb = (long long)prev.s * G.send_cap + (long long)excl_mig;
                if ((long long)excl_mig + (long long)prev.n_mig > G.send_cap) { raise(T.status, -4); sb = -1; }
                sm.sendbase = sb;
                // next ticket: taken only after this look-back has finished, so a CTA never holds an
                // unpublished ticket while it waits on predecessors
                sm.next_ticket = atomicAdd(T.ticket, 1u);
            }
        } else if (!prev.valid && threadIdx.x == 0) {
            sm.next_ticket = atomicAdd(T.ticket, 1u);
        }
        __syncthreads();                                                                                 // B2

        // ============ copy-out of the previous tile: staged order == output order, coalesced ============
        if (prev.valid) {
            const TileBuf& B = buf[b ^ 1];
            const size_t stay_base = (size_t)prev.s * (size_t)G.cap + (size_t)sm.stay_excl;
            const long long sendbase = sm.sendbase;
            for (uint32_t j = threadIdx.x; j < prev.n_stay; j += kBlock) {
                const size_t dst = stay_base + j;
#pragma unroll
                for (int a = 0; a < 7; ++a) st_stream(S.f[a] + dst, B.f[a][j]);
                st_stream(S.id + dst, (int64_t)B.id[j]);
            }
            if (sendbase >= 0) {
                for (uint32_t j = threadIdx.x; j < prev.n_mig; j += kBlock) {
                    const size_t dst = (size_t)sendbase + j;
                    const uint32_t src = prev.n_stay + j;
#pragma unroll
                    for (int a = 0; a < 7; ++a) st_stream(Snd.f[a] + dst, B.f[a][src]);
                    st_stream(Snd.id + dst, (int64_t)B.id[src]);
                }
            }
        }
        __syncthreads();                                                                                 // B3
        prev = cur;
    }
}

// ---------------------------------------------------------------------------------------------
// K2b: per-(subdomain, code) exclusive scan of tile_cnt over the tiles of the subdomain ->
// tile_excl (used by the unpack) and the count table totals cnt[s][c] (a4/a5).  One CTA per s.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_code_scan(Geom G, Tables T)
{
    __shared__ uint32_t s_part[8][32];
    const int s = blockIdx.x;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t cnt_s = T.count[s];
    const int nt = (int)((cnt_s + kTile - 1) / kTile);
    const int chunk = (nt + 7) / 8;
    const int t0 = min(nt, warp * chunk), t1 = min(nt, t0 + chunk);
    const size_t row0 = (size_t)s * G.tiles_per_sub;
    uint32_t sum = 0;
    for (int t = t0; t < t1; ++t) sum += T.tile_cnt[(row0 + t) * 32 + lane];
    s_part[warp][lane] = sum;
    __syncthreads();
    uint32_t run = 0, total = 0;
    for (int w = 0; w < 8; ++w) { const uint32_t v = s_part[w][lane]; if (w < warp) run += v; total += v; }
    for (int t = t0; t < t1; ++t) {
        const uint32_t v = T.tile_cnt[(row0 + t) * 32 + lane];
        T.tile_excl[(row0 + t) * 32 + lane] = run;
        run += v;
    }
    if (warp == 0) T.cnt[s * 32 + lane] = total;
}

// compact tile prefix: tile_start[s] = sum_{s' < s} ceil(count[s'] / kTile); one CTA
__global__ void __launch_bounds__(1024)
k_tile_index(Geom G, Tables T, int commit)
{
    __shared__ uint32_t sh[1024];
    __shared__ uint32_t s_run;
    if (threadIdx.x == 0) s_run = 0;
    __syncthreads();
    const bool ok = *T.status == 0;
    for (int b0 = 0; b0 < G.P; b0 += 1024) {
        const int r = b0 + threadIdx.x;
        uint32_t v = 0;
        if (r < G.P) {
            if (commit && ok) T.count[r] = T.new_count[r];
            v = (T.count[r] + kTile - 1) / kTile;
        }
        sh[threadIdx.x] = v;
        __syncthreads();
        for (int o = 1; o < 1024; o <<= 1) {
            const uint32_t add = threadIdx.x >= (unsigned)o ? sh[threadIdx.x - o] : 0u;
            __syncthreads();
            sh[threadIdx.x] += add;
            __syncthreads();
        }
        const uint32_t incl = sh[threadIdx.x] + s_run;
        if (r < G.P) T.tile_start[r] = incl - v;
        __syncthreads();
        if (threadIdx.x == 1023) s_run = incl;
        __syncthreads();
    }
    if (threadIdx.x == 0) { T.tile_start[G.P] = s_run; *T.ticket = 0u; }
}

// ---------------------------------------------------------------------------------------------
// K3: table scan (a5 at table level).  stay[s], receive offsets in the fixed order (s ascending,
// c ascending), new counts, overflow flag, totals.  One CTA, thread r owns receiver r.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_table(Geom G, Tables T)
{
    __shared__ unsigned long long s_mig, s_tot;
    if (threadIdx.x == 0) { s_mig = 0; s_tot = 0; }
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
