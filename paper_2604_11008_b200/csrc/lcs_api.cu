// lcs_api.cu -- the C ABI of include/lcs.h: argument checks, workspace carving, kernel launches.
// No device allocation happens here (the caller's workspace is carved); every call enqueues on the
// handle's stream.  Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -fmad=false.
#include "../../include/lcs.h"
#include "lcs_kernels.cuh"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <algorithm>
#include <mutex>
#include <new>
#include <vector>

using namespace lcs;

struct lcs_handle {
    Geom G;
    Slabs S, Snd;
    Tables T;
    cudaStream_t stream;
    double* fluid4;           // [N^3][4] repacked fluid (u,v,w,0), in the workspace
    bool have_fluid;
    int64_t* prefix;          // [P+1] scratch for packed copy-out
    void* pool;               // send pool base (also scratch of lcs_set_particles)
    size_t pool_bytes;
    uint32_t epoch;
    bool pushed;              // codes + count table describe a push that has not been migrated
    bool have_particles;
    int sticky;               // last sticky error seen by lcs_get_status
    int64_t launches;
    std::vector<cudaEvent_t>* prof;   // 4 events per recorded step, or null
    int prof_steps, prof_max;
    int grid_fused, grid_pack;         // persistent grid sizes of the tile pass
    CUtensorMap slab_map;              // 2-D view [8 fields][P*cap slots] of the slabs, box 8 x kTile (bulk tile loads)
    bool rk2;                          // the 9 extra arrays of the two-stage RK2 exist (lcs_params.enable_rk2)
    Slabs SB;                          // RK2: x0 y0 z0 k1x k1y k1z + 2 spare arrays (a group of 8 for the tile pass)
    CUtensorMap mapB;
    CUtensorMap map_push_ld, map_push_st;   // the slabs again with a box of 7 rows (x .. d, loads) and of 6 rows (x .. vz, stores)
    size_t gacc_bytes;
    cudaStream_t copy_stream;          // lcs_step_fused_host: the host copies run here, beside the kernels (created on first use)
    cudaEvent_t ev[12];                // start, x/y/z in, all in, one per array out, copies done
    bool have_copy_stream;
};

namespace {

constexpr size_t kAlign = 256;
inline size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

struct Layout {
    size_t slab_f[7], slab_id, slab_code;
    size_t rk2_b;                      // RK2 group B: 8 arrays, stride as the slabs (0 = absent)
    size_t pool, pool_bytes, fluid4;
    size_t count, cnt, recv_off, new_count, desc, gacc, gacc_bytes, tile_start, send_count, chunk_excl, misc, prefix;
    size_t total;
    int tiles_per_sub, chunks_per_sub, lbgroups_per_sub;
    int64_t send_cap;
};

inline size_t brick_records(int N, int Px, int Py, int Pz)
{
    return (size_t)(N / Px + 2) * (size_t)(N / Py + 2) * (size_t)(N / Pz + 2);
}

bool valid_args(int N, int Px, int Py, int Pz, int64_t cap, const lcs_params* prm)
{
    if (!prm) return false;
    if (N < 2 || N > 1623 || Px < 1 || Py < 1 || Pz < 1) return false;   // (N + 2)^3 < 2^32 with one subdomain; the brick test below is the rule
    if (Px > 1024 || Py > 1024 || Pz > 1024) return false;   // packed subdomain coordinates (10 bits each)
    if (N % Px || N % Py || N % Pz) return false;
    const int64_t P = (int64_t)Px * Py * Pz;
    if (P > 8192) return false;                          // grid.y and shared-histogram limits
    if ((unsigned long long)P * brick_records(N, Px, Py, Pz) >= (1ull << 32)) return false;   // fluid record indices are 32-bit
    if (cap < 2 || (cap & 1)) return false;               // even: slab bases stay 16-byte aligned
    if (cap > 0x7fffffff) return false;
    if ((unsigned long long)P * (unsigned long long)cap >= (1ull << 31)) return false;   // slot indices are 32-bit, and the bulk
                                                                                         // tensor copies take SIGNED 32-bit coordinates
    if (prm->send_capacity < 0 || (prm->send_capacity & 1) || prm->send_capacity > cap) return false;
    if (!(prm->nu > 0.0) || !(prm->rho_ratio > 0.0)) return false;
    if (prm->drag_model != 0 && prm->drag_model != 1) return false;
    if (prm->enable_rk2 != 0 && prm->enable_rk2 != 1) return false;
    if (!std::isfinite(prm->g[0]) || !std::isfinite(prm->g[1]) || !std::isfinite(prm->g[2])) return false;
    return true;
}

Layout make_layout(int N, int Px, int Py, int Pz, int64_t cap, const lcs_params* prm)
{
    Layout L;
    const size_t P = (size_t)Px * Py * Pz;
    const size_t slots = P * (size_t)cap;
    L.send_cap = prm->send_capacity ? prm->send_capacity : cap;
    L.tiles_per_sub = (int)((cap + kTile - 1) / kTile);
    L.chunks_per_sub = (int)((L.send_cap + kChunk - 1) / kChunk);
    L.lbgroups_per_sub = (L.tiles_per_sub + 31) / 32;
    const size_t ntiles = P * (size_t)L.tiles_per_sub;
    size_t off = 0;
    for (int a = 0; a < 7; ++a) { L.slab_f[a] = off; off = align_up(off + slots * 8); }
    L.slab_id = off;   off = align_up(off + slots * 8);
    L.slab_code = off; off = align_up(off + slots);
    L.rk2_b = 0;
    if (prm->enable_rk2) { L.rk2_b = off; off += 8 * align_up(slots * 8); }
    // send pool: 8 arrays of P*send_cap slots + one code byte per slot; doubles as lcs_set_particles scratch
    const size_t send_bytes = 8 * align_up(P * (size_t)L.send_cap * 8) + align_up(P * (size_t)L.send_cap);
    const size_t set_tiles = (slots + kSetTile - 1) / kSetTile;
    const size_t set_bytes = align_up(slots * 4) + align_up(set_tiles * P * 4);
    L.pool = off; L.pool_bytes = send_bytes > set_bytes ? send_bytes : set_bytes;
    off = align_up(off + L.pool_bytes);
    // fluid bricks: every subdomain's cells plus a periodic halo of one cell, 32 B per record
    L.fluid4 = off;    off = align_up(off + P * brick_records(N, Px, Py, Pz) * 32);
    L.count = off;     off = align_up(off + P * 4);
    L.cnt = off;       off = align_up(off + P * 32 * 4);
    L.recv_off = off;  off = align_up(off + P * 32 * 4);
    L.new_count = off; off = align_up(off + P * 4);
    L.desc = off;      off = align_up(off + ntiles * 8);
    L.gacc = off;      L.gacc_bytes = P * (size_t)L.lbgroups_per_sub * 8; off = align_up(off + L.gacc_bytes);
    L.tile_start = off; off = align_up(off + (P + 1) * 4);
    L.send_count = off; off = align_up(off + P * 4);
    L.chunk_excl = off; off = align_up(off + P * (size_t)L.chunks_per_sub * 32 * 4);
    L.misc = off;      off = align_up(off + 256);
    L.prefix = off;    off = align_up(off + (P + 1) * 8);
    L.total = off;
    return L;
}

// Tensor map of one group of 8 arrays for the bulk tile loads: 2-D [8 fields][slots] of 8-byte words, rows `stride` bytes
// apart, box 8 x kTile.  The encoder is fetched from the driver through the runtime (no link against libcuda).
bool make_slab_map(CUtensorMap* out, void* base, size_t slots, size_t stride, int rows = 8)
{
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) return false;
    const cuuint64_t gdim[2] = {(cuuint64_t)slots, 8};
    const cuuint64_t gstride[1] = {(cuuint64_t)stride};
    const cuuint32_t box[2] = {(cuuint32_t)kTile, (cuuint32_t)rows};
    const cuuint32_t estr[2] = {1, 1};
    return reinterpret_cast<encode_fn>(fn)(out, CU_TENSOR_MAP_DATA_TYPE_UINT64, 2, base, gdim, gstride, box, estr,
                                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                           CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

inline size_t tile_pass_smem(int P)
{
    return kWarps * kNBuf * (sizeof(TileBuf) + sizeof(uint64_t)) + (P <= kTableSmemMax ? (size_t)(2 * P + 1) * sizeof(uint32_t) : 0);
}

// dynamic shared memory of k_set_scatter with W warps per tile
inline size_t set_scatter_smem(int W, int P)
{
    return ((size_t)(W + 1) * P + 2 * kSetTile + 1) * 2 + (size_t)kSetTile * 4 + 16;
}

// cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the kernel (per device), not to a handle: it is set to the
// largest size any handle can ask for -- the same value on every lcs_create -- so that live handles with different P
// cannot lower it under one another.  Largest tile pass: P = kTableSmemMax (tables mirrored in shared memory); largest
// k_set_scatter: P = 8192 with two warps per tile.
inline void set_kernel_smem_limits()
{
    const int tp = (int)tile_pass_smem(kTableSmemMax);
    auto lim = [tp](auto kernel) { cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, tp); };
    lim(k_tile_pass<0, true, 0>); lim(k_tile_pass<0, false, 0>);
    lim(k_tile_pass<1, true, 0>); lim(k_tile_pass<1, true, 1>); lim(k_tile_pass<1, false, 0>); lim(k_tile_pass<1, false, 1>);
    lim(k_tile_pass<2, true, 0>); lim(k_tile_pass<2, true, 1>); lim(k_tile_pass<2, false, 0>); lim(k_tile_pass<2, false, 1>);
    lim(k_tile_pass<3, true, 0>); lim(k_tile_pass<3, true, 1>); lim(k_tile_pass<3, false, 0>); lim(k_tile_pass<3, false, 1>);
    lim(k_push_tiles<true, 0>); lim(k_push_tiles<true, 1>); lim(k_push_tiles<false, 0>); lim(k_push_tiles<false, 1>);
    cudaFuncSetAttribute(k_set_scatter, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)set_scatter_smem(2, 8192));
}

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

inline int check_launch(lcs_t* h, int n = 1)
{
    h->launches += n;
    return cudaGetLastError() == cudaSuccess ? LCS_OK : LCS_ERR_CUDA;   // consumed: a failed launch on one handle does not
                                                                          // make every later call on every handle fail
}

// One round of the migration machinery on one group of 8 arrays (the slabs, or an RK2 group that travels with the same
// codes): tile pass, per-code scan, table, unpack; `commit` also installs the new counts and the next tile index.  The
// rounds of one migration see the same codes and the same counts, so they apply the same permutation.
int enqueue_tile_pass(lcs_t* h, int mode, double dt, const Slabs* grp = nullptr, const CUtensorMap* map = nullptr,
                      bool commit = true, int nf = 8)
{
    const Geom& G = h->G;
    const Slabs& S = grp ? *grp : h->S;
    const CUtensorMap& M = map ? *map : h->slab_map;
    h->epoch = (h->epoch + 1u) & 0xffffffu;                // 24 bits: the count field of a look-back word
    if (h->epoch == 0u) {                                  // wrapped: no word of 2^24 launches ago may look current
        h->epoch = 1u;
        cudaMemsetAsync(h->T.desc, 0, (size_t)G.P * (size_t)G.tiles_per_sub * 8, h->stream);
    }
    const bool rec = h->prof && h->prof_steps < h->prof_max;
    cudaEvent_t* ev = rec ? h->prof->data() + 4 * h->prof_steps : nullptr;
    if (rec) cudaEventRecord(ev[0], h->stream);
    const size_t smem = tile_pass_smem(G.P);
    const bool big = G.P > kTableSmemMax;
    const bool fused = mode != 0;
    const bool sn = fused && G.drag_model == 1;            // the unfused pass carries no push: one instantiation
#define LCS_LAUNCH_TP(F, B, D, GRID) \
    k_tile_pass<F, B, D><<<GRID, kBlock, smem, h->stream>>>(G, S, h->Snd, h->T, h->fluid4, dt, h->epoch, M, h->SB, nf)
#define LCS_LAUNCH_MODE(F) \
    do { if (big) { if (sn) LCS_LAUNCH_TP(F, true, 1, h->grid_fused); else LCS_LAUNCH_TP(F, true, 0, h->grid_fused); } \
         else     { if (sn) LCS_LAUNCH_TP(F, false, 1, h->grid_fused); else LCS_LAUNCH_TP(F, false, 0, h->grid_fused); } } while (0)
    if (mode == 1) LCS_LAUNCH_MODE(1);
    else if (mode == 2) LCS_LAUNCH_MODE(2);
    else if (mode == 3) LCS_LAUNCH_MODE(3);
    else {
        if (big) LCS_LAUNCH_TP(0, true, 0, h->grid_pack); else LCS_LAUNCH_TP(0, false, 0, h->grid_pack);
    }
#undef LCS_LAUNCH_MODE
#undef LCS_LAUNCH_TP
    if (rec) cudaEventRecord(ev[1], h->stream);
    k_send_scan<<<G.P, 32 * kScanWarps, 0, h->stream>>>(G, h->Snd, h->T);
    k_table<<<(G.P + 7) / 8, 256, 0, h->stream>>>(G, h->T);
    if (rec) cudaEventRecord(ev[2], h->stream);
    k_unpack<<<dim3((G.chunks_per_sub + kUnpackWarps - 1) / kUnpackWarps, G.P), 32 * kUnpackWarps, 0, h->stream>>>(G, S, h->Snd, h->T, nf);
    k_tile_index<<<1, 1024, 0, h->stream>>>(G, h->T, commit ? 1 : 0);     // (also resets the tile ticket and the look-back accumulators for the next round)
    if (rec) { cudaEventRecord(ev[3], h->stream); ++h->prof_steps; }
    if (commit) h->pushed = false;
    return check_launch(h, 5);
}

// Cells per axis of the pair count's cell list (lcs_pair_count, lcs_pair_count_static).  The walk over the 27 neighbouring
// cells finds every partner closer than r_hi only if the cell side L/M is LARGER than r_hi by more than the rounding of
// the cell index (a * M/L, floored): with L/M == r_hi up to rounding (lattice data, r_hi = L/M) two particles that count
// can sit two cells apart.  So M = floor(L / (r_hi (1 + 1e-12))), except that with three cells per axis the 27
// neighbours are the whole box and any side will do (r_hi = L/3 lands there).  Then: about one particle per cell, at
// most 400 per axis (15,625 scan chunks; k_scan_top takes 16,384), and whatever fits `avail` bytes of scratch.
long long pair_cells_per_axis(double L, double r_hi, size_t slots, size_t avail)
{
    long long M = std::max<long long>(3, std::min<long long>(400, (long long)std::floor(L / (r_hi * (1.0 + 1e-12)))));
    M = std::min<long long>(M, std::max<long long>(3, (long long)std::cbrt((double)slots)));
    while (M > 3 && (size_t)(8 * M * M * M + 4 + 4 * ((M * M * M + kScanChunk - 1) / kScanChunk) + 256) > avail) --M;
    if ((size_t)(8 * M * M * M + 4 + 4 * ((M * M * M + kScanChunk - 1) / kScanChunk) + 256) > avail) return 0;
    return M;
}

}  // namespace

extern "C" {

const char* lcs_version(void) { return "lcs_b200 0.2 sm_100a"; }

size_t lcs_staging_bytes(int64_t n, int P)
{
    if (n < 0 || P < 1) return 0;
    return 8 * align_up((size_t)n * 8) + align_up((size_t)P * 8);
}

size_t lcs_workspace_bytes(int N, int Px, int Py, int Pz, int64_t capacity, const lcs_params* prm)
{
    if (!valid_args(N, Px, Py, Pz, capacity, prm)) return 0;
    return make_layout(N, Px, Py, Pz, capacity, prm).total;
}

int lcs_create(int N, int Px, int Py, int Pz, int64_t capacity, const lcs_params* prm, void* d_workspace,
               size_t workspace_bytes, void* cuda_stream, lcs_t** out)
{
    if (!out) return LCS_ERR_INVALID_ARG;
    *out = nullptr;
    if (!valid_args(N, Px, Py, Pz, capacity, prm) || !d_workspace) return LCS_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(d_workspace) % kAlign) return LCS_ERR_INVALID_ARG;
    const Layout L = make_layout(N, Px, Py, Pz, capacity, prm);
    if (workspace_bytes < L.total) return LCS_ERR_INVALID_ARG;
    lcs_t* h = new (std::nothrow) lcs_handle();
    if (!h) return LCS_ERR_NOMEM;
    std::memset(static_cast<void*>(h), 0, sizeof(*h));
    Geom& G = h->G;
    G.N = N; G.Px = Px; G.Py = Py; G.Pz = Pz; G.P = Px * Py * Pz;
    G.nx = N / Px; G.ny = N / Py; G.nz = N / Pz;
    G.bj = G.nz + 2; G.bi = (G.ny + 2) * (G.nz + 2);
    G.brick = (uint32_t)brick_records(N, Px, Py, Pz);
    G.tiles_per_sub = L.tiles_per_sub;
    G.chunks_per_sub = L.chunks_per_sub;
    G.lbgroups_per_sub = L.lbgroups_per_sub;
    G.cap = capacity; G.send_cap = L.send_cap;
    // all doubles are computed once on the host and passed as data (rule R6)
    G.L = 6.283185307179586;                      // 2*pi*L0, L0 = 1
    G.inv_dx = (double)N / G.L;
    G.K_tau = prm->rho_ratio / (18.0 * prm->nu);  // tau_p = K_tau * d^2
    G.L_below = std::nextafter(G.L, 0.0);
    G.gx = prm->g[0]; G.gy = prm->g[1]; G.gz = prm->g[2];
    G.inv_nu = 1.0 / prm->nu;
    G.drag_model = prm->drag_model;
    char* w = static_cast<char*>(d_workspace);
    const size_t P = (size_t)G.P;
    for (int a = 0; a < 7; ++a) h->S.f[a] = reinterpret_cast<double*>(w + L.slab_f[a]);
    h->S.id = reinterpret_cast<int64_t*>(w + L.slab_id);
    h->S.code = reinterpret_cast<uint8_t*>(w + L.slab_code);
    h->pool = w + L.pool; h->pool_bytes = L.pool_bytes;
    const size_t send_arr = align_up(P * (size_t)L.send_cap * 8);
    for (int a = 0; a < 7; ++a) h->Snd.f[a] = reinterpret_cast<double*>(w + L.pool + a * send_arr);
    h->Snd.id = reinterpret_cast<int64_t*>(w + L.pool + 7 * send_arr);
    h->Snd.code = reinterpret_cast<uint8_t*>(w + L.pool + 8 * send_arr);
    h->fluid4 = reinterpret_cast<double*>(w + L.fluid4);
    h->T.count = reinterpret_cast<uint32_t*>(w + L.count);
    h->T.cnt = reinterpret_cast<uint32_t*>(w + L.cnt);
    h->T.recv_off = reinterpret_cast<uint32_t*>(w + L.recv_off);
    h->T.new_count = reinterpret_cast<uint32_t*>(w + L.new_count);
    h->T.desc = reinterpret_cast<uint64_t*>(w + L.desc);
    h->T.gacc = reinterpret_cast<unsigned long long*>(w + L.gacc);
    h->gacc_bytes = L.gacc_bytes;
    h->T.tile_start = reinterpret_cast<uint32_t*>(w + L.tile_start);
    h->T.send_count = reinterpret_cast<uint32_t*>(w + L.send_count);
    h->T.chunk_excl = reinterpret_cast<uint32_t*>(w + L.chunk_excl);
    h->T.ticket = reinterpret_cast<unsigned int*>(w + L.misc);
    h->T.status = reinterpret_cast<int*>(w + L.misc + 16);
    h->T.n_migrated = reinterpret_cast<unsigned long long*>(w + L.misc + 32);
    h->T.n_total = reinterpret_cast<unsigned long long*>(w + L.misc + 48);
    h->prefix = reinterpret_cast<int64_t*>(w + L.prefix);
    h->stream = static_cast<cudaStream_t>(cuda_stream);
    if (!make_slab_map(&h->slab_map, w + L.slab_f[0], (size_t)P * (size_t)capacity, L.slab_f[1] - L.slab_f[0])) { delete h; return LCS_ERR_CUDA; }
    if (!make_slab_map(&h->map_push_ld, w + L.slab_f[0], (size_t)P * (size_t)capacity, L.slab_f[1] - L.slab_f[0], 7) ||
        !make_slab_map(&h->map_push_st, w + L.slab_f[0], (size_t)P * (size_t)capacity, L.slab_f[1] - L.slab_f[0], 6)) { delete h; return LCS_ERR_CUDA; }
    h->rk2 = prm->enable_rk2 == 1;
    if (h->rk2) {   // the RK2 group: same stride and shape as the slabs, so the same tile pass moves it
        const size_t st = L.slab_f[1] - L.slab_f[0];
        for (int a = 0; a < 7; ++a) h->SB.f[a] = reinterpret_cast<double*>(w + L.rk2_b + a * st);
        h->SB.id = reinterpret_cast<int64_t*>(w + L.rk2_b + 7 * st);
        h->SB.code = h->S.code;
        if (!make_slab_map(&h->mapB, w + L.rk2_b, (size_t)P * (size_t)capacity, st, 6)) { delete h; return LCS_ERR_CUDA; }
        if (cudaMemsetAsync(w + L.rk2_b, 0, 8 * st, h->stream) != cudaSuccess) { delete h; return LCS_ERR_CUDA; }
    }
    {   // persistent grids: one wave of resident CTAs
        int dev = 0, sms = 0, occ_f = 0, occ_p = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        const size_t smem = tile_pass_smem(G.P);
        set_kernel_smem_limits();
        auto setup = [&](auto kernel, int& occ) {
            int o = 0;
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, kernel, kBlock, smem);
            occ = occ == 0 ? o : std::min(occ, o);
        };
        if (G.P > kTableSmemMax) {
            setup(k_tile_pass<1, true, 0>, occ_f); setup(k_tile_pass<1, true, 1>, occ_f);
            setup(k_tile_pass<2, true, 0>, occ_f); setup(k_tile_pass<2, true, 1>, occ_f);
            setup(k_tile_pass<3, true, 0>, occ_f); setup(k_tile_pass<3, true, 1>, occ_f);
            setup(k_tile_pass<0, true, 0>, occ_p);
            setup(k_push_tiles<true, 0>, occ_f); setup(k_push_tiles<true, 1>, occ_f);
        } else {
            setup(k_tile_pass<1, false, 0>, occ_f); setup(k_tile_pass<1, false, 1>, occ_f);
            setup(k_tile_pass<2, false, 0>, occ_f); setup(k_tile_pass<2, false, 1>, occ_f);
            setup(k_tile_pass<3, false, 0>, occ_f); setup(k_tile_pass<3, false, 1>, occ_f);
            setup(k_tile_pass<0, false, 0>, occ_p);
            setup(k_push_tiles<false, 0>, occ_f); setup(k_push_tiles<false, 1>, occ_f);
        }
        if (sms < 1) sms = 148;
        const long long max_tiles = ((long long)G.P * G.tiles_per_sub + kWarps - 1) / kWarps;
        h->grid_fused = (int)std::min<long long>(max_tiles, (long long)sms * (occ_f > 0 ? occ_f : 1));
        h->grid_pack = (int)std::min<long long>(max_tiles, (long long)sms * (occ_p > 0 ? occ_p : 1));
    }
    // tables start at zero (epoch 0 is never published; counts empty)
    if (cudaMemsetAsync(w + L.count, 0, L.total - L.count, h->stream) != cudaSuccess) { delete h; return LCS_ERR_CUDA; }
    *out = h;
    return LCS_OK;
}

int lcs_destroy(lcs_t* h)
{
    if (!h) return LCS_ERR_INVALID_ARG;
    cudaStreamSynchronize(h->stream);
    if (h->prof) lcs_profile_end(h, nullptr, nullptr, nullptr, nullptr);
    if (h->have_copy_stream) {
        cudaStreamSynchronize(h->copy_stream);
        for (auto& e : h->ev) cudaEventDestroy(e);
        cudaStreamDestroy(h->copy_stream);
    }
    delete h;
    return LCS_OK;
}

int lcs_set_fluid(lcs_t* h, const double* d_u, const double* d_v, const double* d_w)
{
    if (!h || !d_u || !d_v || !d_w) return LCS_ERR_INVALID_ARG;
    if (!aligned16(d_u) || !aligned16(d_v) || !aligned16(d_w)) return LCS_ERR_INVALID_ARG;
    const Geom& G = h->G;
    // chunks of the local (a, c) plane: as equal as possible, at most kRpA x kRpC
    const int ea = G.nx + 2, ec = G.nz + 2;
    const int na = (ea + kRpA - 1) / kRpA, nc = (ec + kRpC - 1) / kRpC;
    const int ca = (ea + na - 1) / na, cc = (ec + nc - 1) / nc;
    k_repack_fluid<<<dim3(na * nc, G.ny + 2, G.P), 256, 0, h->stream>>>(G, d_u, d_v, d_w, h->fluid4, ca, cc, na);
    h->have_fluid = true;
    return check_launch(h);
}

static int set_particles_impl(lcs_t* h, int64_t n, const double* d_x, const double* d_y, const double* d_z,
                              const double* d_vx, const double* d_vy, const double* d_vz, const double* d_diam,
                              const int64_t* d_id, cudaEvent_t rest_ready)
{   // rest_ready (may be null): an event after which d_vx .. d_id are valid; owner, scan and tile index need x, y, z only
    if (!h || n < 0) return LCS_ERR_INVALID_ARG;
    const Geom& G = h->G;
    if (n > (int64_t)G.P * G.cap) return LCS_ERR_INVALID_ARG;
    if (n > 0 && (!d_x || !d_y || !d_z || !d_vx || !d_vy || !d_vz || !d_diam || !d_id)) return LCS_ERR_INVALID_ARG;
    if (!aligned16(d_x) || !aligned16(d_y) || !aligned16(d_z) || !aligned16(d_vx) || !aligned16(d_vy) || !aligned16(d_vz) ||
        !aligned16(d_diam) || !aligned16(d_id)) return LCS_ERR_INVALID_ARG;
    // a fresh particle set clears the sticky error
    h->sticky = 0;
    h->pushed = false;
    h->have_particles = true;
    cudaMemsetAsync(h->T.status, 0, sizeof(int), h->stream);
    cudaMemsetAsync(h->T.n_migrated, 0, sizeof(unsigned long long), h->stream);
    const int ntiles = (int)((n + kSetTile - 1) / kSetTile);
    int32_t* owner = static_cast<int32_t*>(h->pool);
    uint32_t* tilehist = reinterpret_cast<uint32_t*>(static_cast<char*>(h->pool) + align_up((size_t)G.P * (size_t)G.cap * 4));
    if (ntiles > 0)
        k_set_owner<<<ntiles, 256, (size_t)G.P * 4, h->stream>>>(G, h->T, n, d_x, d_y, d_z, owner, tilehist);
    k_set_scan<<<(G.P + 31) / 32, 1024, 0, h->stream>>>(G, h->T, ntiles, tilehist, n);
    k_tile_index<<<1, 1024, 0, h->stream>>>(G, h->T, 0);
    if (rest_ready) cudaStreamWaitEvent(h->stream, rest_ready, 0);
    if (ntiles > 0) {
        int W = 8;                                                           // warps per tile, a power of two: W * P 16-bit
        while (W > 1 && W * G.P > 16384) W >>= 1;                             // counters in shared memory
        const size_t smem = set_scatter_smem(W, G.P);        // within the limit lcs_create set (set_kernel_smem_limits)
        InPtrs I;
        I.f[0] = d_x; I.f[1] = d_y; I.f[2] = d_z; I.f[3] = d_vx; I.f[4] = d_vy; I.f[5] = d_vz; I.f[6] = d_diam;
        I.id = d_id;
        k_set_scatter<<<ntiles, 32 * W, smem, h->stream>>>(G, h->S, n, I, owner, tilehist, W);
    }
    return check_launch(h, ntiles > 0 ? 4 : 2);
}

int lcs_set_particles(lcs_t* h, int64_t n, const double* d_x, const double* d_y, const double* d_z,
                      const double* d_vx, const double* d_vy, const double* d_vz, const double* d_diam,
                      const int64_t* d_id)
{
    return set_particles_impl(h, n, d_x, d_y, d_z, d_vx, d_vy, d_vz, d_diam, d_id, nullptr);
}

int lcs_particle_step(lcs_t* h, double dt)
{
    if (!h || !(dt > 0.0) || !std::isfinite(dt)) return LCS_ERR_INVALID_ARG;
    if (!h->have_fluid || !h->have_particles || h->pushed) return LCS_ERR_STATE;   // a pending push must be migrated first
    if (h->sticky) return h->sticky;
    const Geom& G = h->G;
    cudaMemsetAsync(h->T.cnt, 0, (size_t)G.P * 32 * 4, h->stream);
    {
        const size_t smem = tile_pass_smem(G.P);
        const bool big = G.P > kTableSmemMax, sn = G.drag_model == 1;
#define LCS_LAUNCH_PUSH(B, D) \
    k_push_tiles<B, D><<<h->grid_fused, kBlock, smem, h->stream>>>(G, h->S, h->T, h->fluid4, dt, h->map_push_ld, h->map_push_st)
        if (big) { if (sn) LCS_LAUNCH_PUSH(true, 1); else LCS_LAUNCH_PUSH(true, 0); }
        else     { if (sn) LCS_LAUNCH_PUSH(false, 1); else LCS_LAUNCH_PUSH(false, 0); }
#undef LCS_LAUNCH_PUSH
    }
    h->pushed = true;
    return check_launch(h);
}

int lcs_migrate(lcs_t* h)
{
    if (!h) return LCS_ERR_INVALID_ARG;
    if (!h->pushed) return LCS_ERR_STATE;
    if (h->sticky) return h->sticky;
    return enqueue_tile_pass(h, 0, 0.0);
}

int lcs_migrate_sweeps(lcs_t* h)
{
    if (!h) return LCS_ERR_INVALID_ARG;
    if (!h->have_particles) return LCS_ERR_STATE;
    if (h->sticky) return h->sticky;
    const Geom& G = h->G;
    for (int axis = 0; axis < 3; ++axis) {
        k_classify_axis<<<dim3((unsigned)((G.cap + 1023) / 1024), G.P), 256, 0, h->stream>>>(G, h->S.f[axis], h->S.code, h->T.count,
                                                                                                h->T.status, axis);
        int rc = check_launch(h);
        if (rc == LCS_OK) rc = enqueue_tile_pass(h, 0, 0.0);
        if (rc != LCS_OK) return rc;
    }
    return LCS_OK;
}

int lcs_step_rk2(lcs_t* h, double dt)
{
    if (!h || !(dt > 0.0) || !std::isfinite(dt)) return LCS_ERR_INVALID_ARG;
    if (!h->rk2 || !h->have_fluid || !h->have_particles || h->pushed) return LCS_ERR_STATE;
    if (h->sticky) return h->sticky;
    // Stage 1 runs inside the tile pass of the slabs (X1, V0, d, id migrate; X0, K1 and the code byte are written at the
    // particle's slot), then group B (X0, K1) travels in an unfused round with the same codes, which commits the counts.
    int rc = enqueue_tile_pass(h, 2, dt, &h->S, &h->slab_map, false);
    if (rc == LCS_OK) rc = enqueue_tile_pass(h, 0, 0.0, &h->SB, &h->mapB, true, 6);     // X0, K1: six live arrays
    if (rc != LCS_OK) return rc;
    // Stage 2 runs inside the tile pass too: it reads X0, K1 of group B at the particle's slot; only X, V, d, id are live
    // afterwards, so this one round ends the step.
    return enqueue_tile_pass(h, 3, dt);
}

int lcs_step_fused(lcs_t* h, double dt)
{
    if (!h || !(dt > 0.0) || !std::isfinite(dt)) return LCS_ERR_INVALID_ARG;
    if (!h->have_fluid || !h->have_particles || h->pushed) return LCS_ERR_STATE;   // a pending push must be migrated first
    if (h->sticky) return h->sticky;
    return enqueue_tile_pass(h, 1, dt);
}

int lcs_get_counts(lcs_t* h, int64_t* d_counts)
{
    if (!h || !d_counts) return LCS_ERR_INVALID_ARG;
    k_counts_out<<<1, 256, 0, h->stream>>>(h->G, h->T, d_counts, nullptr);
    return check_launch(h);
}

static int copy_out(lcs_t* h, int64_t* d_counts, OutPtrs O)
{
    const Geom& G = h->G;
    k_counts_out<<<1, 256, 0, h->stream>>>(G, h->T, d_counts, h->prefix);
    k_copy_out<<<dim3((unsigned)((G.cap + kCopyTile - 1) / kCopyTile), G.P), 256, 0, h->stream>>>(G, h->S, h->T, h->prefix, O, h->pushed ? 1 : 0);
    return check_launch(h, 2);
}

int lcs_get_particles(lcs_t* h, int64_t* d_counts, double* d_x, double* d_y, double* d_z, double* d_vx,
                      double* d_vy, double* d_vz, double* d_diam, int64_t* d_id)
{
    if (!h) return LCS_ERR_INVALID_ARG;
    if (!aligned16(d_counts) || !aligned16(d_x) || !aligned16(d_y) || !aligned16(d_z) || !aligned16(d_vx) || !aligned16(d_vy) ||
        !aligned16(d_vz) || !aligned16(d_diam) || !aligned16(d_id)) return LCS_ERR_INVALID_ARG;      // NULL (= skip) is aligned
    OutPtrs O;
    O.f[0] = d_x; O.f[1] = d_y; O.f[2] = d_z; O.f[3] = d_vx; O.f[4] = d_vy; O.f[5] = d_vz; O.f[6] = d_diam;
    O.id = d_id; O.code = nullptr;
    return copy_out(h, d_counts, O);
}

int lcs_get_codes(lcs_t* h, uint8_t* d_codes)
{
    if (!h || !d_codes) return LCS_ERR_INVALID_ARG;
    OutPtrs O;
    for (int a = 0; a < 7; ++a) O.f[a] = nullptr;
    O.id = nullptr; O.code = d_codes;
    return copy_out(h, nullptr, O);
}

int lcs_get_count_table(lcs_t* h, int64_t* d_table)
{
    if (!h || !d_table) return LCS_ERR_INVALID_ARG;
    const int n = h->G.P * kNC;
    k_table_out<<<(n + 255) / 256, 256, 0, h->stream>>>(h->G, h->T, d_table, h->pushed ? 1 : 0);
    return check_launch(h);
}

int lcs_pair_count(lcs_t* h, double r_lo, double r_hi, int64_t* d_count)
{
    if (!h || !d_count || (reinterpret_cast<uintptr_t>(d_count) & 7u)) return LCS_ERR_INVALID_ARG;
    if (!(r_lo >= 0.0) || !(r_hi > r_lo) || !std::isfinite(r_hi)) return LCS_ERR_INVALID_ARG;
    const Geom& G = h->G;
    if (r_hi > G.L / 3.0) return LCS_ERR_INVALID_ARG;          // the cell list needs at least three cells per axis
    if (!h->have_particles || h->pushed) return LCS_ERR_STATE;
    if (h->sticky) return h->sticky;
    // scratch in the send pool (free between steps): the positions sorted by cell (three arrays), then the cell arrays
    const size_t slots = (size_t)G.P * (size_t)G.cap;
    const size_t arr_bytes = align_up(slots * 8);
    const size_t idx_bytes = 3 * arr_bytes;
    if (h->pool_bytes < idx_bytes + 1024) return LCS_ERR_INVALID_ARG;
    const size_t avail = h->pool_bytes - idx_bytes;
    const long long M = pair_cells_per_axis(G.L, r_hi, slots, avail);
    if (M < 3) return LCS_ERR_INVALID_ARG;
    const size_t ncell = (size_t)(M * M * M);
    const int nchunks = (int)((ncell + kScanChunk - 1) / kScanChunk);
    char* base = static_cast<char*>(h->pool);
    double* sx = reinterpret_cast<double*>(base);
    double* sy = reinterpret_cast<double*>(base + arr_bytes);
    double* sz = reinterpret_cast<double*>(base + 2 * arr_bytes);
    uint32_t* cellstart = reinterpret_cast<uint32_t*>(base + idx_bytes);       // [ncell + 1]
    uint32_t* cellfill = cellstart + ncell + 1;                                // [ncell]
    uint32_t* sums = cellfill + ncell;                                         // [nchunks]
    PairGeom Q;
    Q.M = (int)M; Q.inv_cell = (double)M / G.L; Q.L = G.L; Q.half_L = 0.5 * G.L; Q.lo2 = r_lo * r_lo; Q.hi2 = r_hi * r_hi;
    cudaMemsetAsync(cellstart, 0, (2 * ncell + 1) * 4, h->stream);
    cudaMemsetAsync(d_count, 0, 8, h->stream);
    const dim3 pgrid((unsigned)((G.cap + 255) / 256), G.P);
    k_pc_count<<<pgrid, 256, 0, h->stream>>>(G, h->S, h->T, Q, cellstart);
    k_scan_sums<<<nchunks, 256, 0, h->stream>>>(cellstart, ncell, sums);
    k_scan_top<<<1, 1024, 0, h->stream>>>(sums, nchunks, cellstart + ncell);
    k_scan_apply<<<nchunks, 256, 0, h->stream>>>(cellstart, ncell, sums);
    k_pc_fill<<<pgrid, 256, 0, h->stream>>>(G, h->S, h->T, Q, cellstart, cellfill, sx, sy, sz);
    k_pc_pairs<<<(unsigned)((slots + 255) / 256), 256, 0, h->stream>>>(Q, cellstart, sx, sy, sz, cellstart + ncell,
                                                                        reinterpret_cast<unsigned long long*>(d_count));
    return check_launch(h, 6);
}

int lcs_get_status(lcs_t* h, int* sticky_error, int64_t* n_total, int64_t* n_migrated_last)
{
    if (!h) return LCS_ERR_INVALID_ARG;
    struct { int status; unsigned long long mig, tot; } host;
    if (cudaMemcpyAsync(&host.status, h->T.status, sizeof(int), cudaMemcpyDeviceToHost, h->stream) != cudaSuccess ||
        cudaMemcpyAsync(&host.mig, h->T.n_migrated, 8, cudaMemcpyDeviceToHost, h->stream) != cudaSuccess ||
        cudaMemcpyAsync(&host.tot, h->T.n_total, 8, cudaMemcpyDeviceToHost, h->stream) != cudaSuccess ||
        cudaStreamSynchronize(h->stream) != cudaSuccess) {
        return LCS_ERR_CUDA;
    }
    h->sticky = host.status;
    if (sticky_error) *sticky_error = host.status;
    if (n_total) *n_total = (int64_t)host.tot;
    if (n_migrated_last) *n_migrated_last = (int64_t)host.mig;
    return host.status;
}

int lcs_step_fused_host(lcs_t* h, double dt, int64_t n, const void* const h_in[8], void* const h_out[8],
                        int64_t* h_counts, void* d_staging, size_t staging_bytes)
{
    if (!h || !h_in || !h_out || !h_counts || !d_staging || n < 0) return LCS_ERR_INVALID_ARG;
    const size_t arr = align_up((size_t)n * 8);
    if (staging_bytes < lcs_staging_bytes(n, h->G.P)) return LCS_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(h_counts) & 7u) return LCS_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(d_staging) % kAlign) return LCS_ERR_INVALID_ARG;
    char* st = static_cast<char*>(d_staging);
    for (int a = 0; a < 8; ++a) {
        if (!h_in[a] || !h_out[a]) return LCS_ERR_INVALID_ARG;
        if ((reinterpret_cast<uintptr_t>(h_in[a]) | reinterpret_cast<uintptr_t>(h_out[a])) & 7u) return LCS_ERR_INVALID_ARG;
    }
    // The host copies run on a stream of their own, ordered against the kernels by events, one array at a time: the
    // owner / scan kernels (x, y, z only) run under the copy-in of the other five arrays, and the copy-out of array a
    // runs under the packing of array a+1.  The two directions cannot overlap: the step needs every particle.
    if (!h->have_copy_stream) {
        if (cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); return LCS_ERR_CUDA; }
        int made = 0;
        while (made < 12 && cudaEventCreateWithFlags(&h->ev[made], cudaEventDisableTiming) == cudaSuccess) ++made;
        if (made < 12) {                                        // nothing half-made is left behind
            cudaGetLastError();
            while (made > 0) cudaEventDestroy(h->ev[--made]);
            cudaStreamDestroy(h->copy_stream);
            return LCS_ERR_CUDA;
        }
        h->have_copy_stream = true;
    }
    cudaStream_t cs = h->copy_stream;
    cudaEvent_t ev_start = h->ev[0], ev_xyz = h->ev[1], ev_all = h->ev[2], ev_done = h->ev[11];
    cudaEventRecord(ev_start, h->stream);                       // earlier work on the handle's stream (staging reuse) comes first
    cudaStreamWaitEvent(cs, ev_start, 0);
    for (int a = 0; a < 8; ++a) {
        if (cudaMemcpyAsync(st + a * arr, h_in[a], (size_t)n * 8, cudaMemcpyHostToDevice, cs) != cudaSuccess) return LCS_ERR_CUDA;
        if (a == 2) cudaEventRecord(ev_xyz, cs);
    }
    cudaEventRecord(ev_all, cs);
    double* f[7];
    for (int a = 0; a < 7; ++a) f[a] = reinterpret_cast<double*>(st + a * arr);
    int64_t* ids = reinterpret_cast<int64_t*>(st + 7 * arr);
    int64_t* d_counts = reinterpret_cast<int64_t*>(st + 8 * arr);
    cudaStreamWaitEvent(h->stream, ev_xyz, 0);
    int rc = set_particles_impl(h, n, f[0], f[1], f[2], f[3], f[4], f[5], f[6], ids, ev_all);
    if (rc) return rc;
    rc = lcs_step_fused(h, dt);
    if (rc) return rc;
    // packed copy-out, one array per launch, each followed by its device-to-host copy on the copy stream
    const Geom& G = h->G;
    k_counts_out<<<1, 256, 0, h->stream>>>(G, h->T, d_counts, h->prefix);
    const dim3 cgrid((unsigned)((G.cap + kCopyTile - 1) / kCopyTile), G.P);
    for (int a = 0; a < 8; ++a) {
        OutPtrs O;
        for (int q = 0; q < 7; ++q) O.f[q] = (q == a) ? f[q] : nullptr;
        O.id = (a == 7) ? ids : nullptr; O.code = nullptr;
        k_copy_out<<<cgrid, 256, 0, h->stream>>>(G, h->S, h->T, h->prefix, O, 0);
        cudaEventRecord(h->ev[3 + a], h->stream);
        cudaStreamWaitEvent(cs, h->ev[3 + a], 0);
        if (cudaMemcpyAsync(h_out[a], st + a * arr, (size_t)n * 8, cudaMemcpyDeviceToHost, cs) != cudaSuccess) return LCS_ERR_CUDA;
        if (a == 0 && cudaMemcpyAsync(h_counts, d_counts, (size_t)G.P * 8, cudaMemcpyDeviceToHost, cs) != cudaSuccess) return LCS_ERR_CUDA;
    }
    cudaEventRecord(ev_done, cs);
    cudaStreamWaitEvent(h->stream, ev_done, 0);
    rc = check_launch(h, 9);
    if (rc) return rc;
    return lcs_get_status(h, nullptr, nullptr, nullptr);
}

int lcs_profile_begin(lcs_t* h, int max_steps)
{
    if (!h || max_steps < 1 || max_steps > 4096) return LCS_ERR_INVALID_ARG;
    if (h->prof) lcs_profile_end(h, nullptr, nullptr, nullptr, nullptr);
    h->prof = new (std::nothrow) std::vector<cudaEvent_t>(4 * (size_t)max_steps);
    if (!h->prof) return LCS_ERR_CUDA;
    for (auto& e : *h->prof)
        if (cudaEventCreate(&e) != cudaSuccess) return LCS_ERR_CUDA;
    h->prof_steps = 0; h->prof_max = max_steps;
    return LCS_OK;
}

int lcs_profile_end(lcs_t* h, double* ms_tile_pass, double* ms_table, double* ms_unpack, int* n_steps)
{
    if (!h || !h->prof) return LCS_ERR_STATE;
    int rc = cudaStreamSynchronize(h->stream) == cudaSuccess ? LCS_OK : LCS_ERR_CUDA;
    double acc[3] = {0.0, 0.0, 0.0};
    for (int i = 0; i < h->prof_steps && rc == LCS_OK; ++i)
        for (int k = 0; k < 3; ++k) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, (*h->prof)[4 * i + k], (*h->prof)[4 * i + k + 1]) != cudaSuccess) rc = LCS_ERR_CUDA;
            acc[k] += ms;
        }
    if (ms_tile_pass) *ms_tile_pass = acc[0];
    if (ms_table) *ms_table = acc[1];
    if (ms_unpack) *ms_unpack = acc[2];
    if (n_steps) *n_steps = h->prof_steps;
    for (auto& e : *h->prof) cudaEventDestroy(e);
    delete h->prof;
    h->prof = nullptr; h->prof_steps = 0; h->prof_max = 0;
    return rc;
}

int lcs_probe_gather(lcs_t* h, double window_mb, int iters, double* h_ms, double* h_bytes)
{
    if (!h || !h_ms || !h_bytes || !(window_mb > 0.0) || iters < 1) return LCS_ERR_INVALID_ARG;
    if (!h->have_fluid) return LCS_ERR_STATE;
    const size_t nrec = (size_t)h->G.P * h->G.brick;
    const uint32_t wrecs = (uint32_t)std::max<size_t>(2, std::min<size_t>(nrec, (size_t)(window_mb * 1048576.0 / 32.0)));
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return LCS_ERR_CUDA;
    double* sink = reinterpret_cast<double*>(h->T.n_total) + 8;              // spare words of the misc block
    k_probe_gather<<<sms, 384, 0, h->stream>>>(h->fluid4, wrecs, std::max(1, iters / 8), sink);      // warm-up: fills L2
    cudaEventRecord(e0, h->stream);
    k_probe_gather<<<sms, 384, 0, h->stream>>>(h->fluid4, wrecs, iters, sink);
    cudaEventRecord(e1, h->stream);
    int rc = cudaEventSynchronize(e1) == cudaSuccess ? LCS_OK : LCS_ERR_CUDA;
    float ms = 0.f;
    if (rc == LCS_OK && cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) rc = LCS_ERR_CUDA;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    *h_ms = ms;
    *h_bytes = (double)sms * 384.0 * (double)iters * 8.0 * 32.0;            // one 32-byte sector per load
    h->launches += 2;
    return rc;
}

int64_t lcs_kernel_launches(lcs_t* h) { return h ? h->launches : 0; }

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// lcs_pair_count_static: the pair count for a caller that cannot lend scratch and must not allocate (include/lcs.h has
// the full story: a diagnostics hook inside a time loop whose host application owns all device memory and bans
// cudaMalloc / cudaFree there, with a send pool too small for lcs_pair_count).  The kernels are lcs_pair_count's own;
// only the place of the scratch differs: the array below, which belongs to the library's device image.
//
// g_pc_static is a DEVICE array.  Seen from host code its name is only a handle the runtime knows the array by: taking
// its address on the host yields a host address, and a kernel handed that address faults (or scribbles over host memory
// on systems where the GPU can reach it).  The usable pointer comes from cudaGetSymbolAddress, asked once per device
// with that device current, because every GPU that loads this image has its own copy at its own address.
// ---------------------------------------------------------------------------------------------
namespace {

static __device__ __align__(256) unsigned char g_pc_static[LCS_PAIR_COUNT_STATIC_BYTES];

std::mutex g_pc_static_lock;
void* g_pc_static_ptr[LCS_PAIR_COUNT_STATIC_MAX_DEVICES];     // device address of g_pc_static on device d, or null

// Device address of g_pc_static on the current device (set-up on the first call per device); null on failure.
void* pc_static_scratch(int* dev_out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= LCS_PAIR_COUNT_STATIC_MAX_DEVICES) return nullptr;
    *dev_out = dev;
    std::lock_guard<std::mutex> guard(g_pc_static_lock);
    if (!g_pc_static_ptr[dev]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_pc_static) != cudaSuccess || !p) {
            cudaGetLastError();                                // the failure is reported by the return value
            return nullptr;
        }
        g_pc_static_ptr[dev] = p;
    }
    return g_pc_static_ptr[dev];
}

}  // namespace

extern "C" int lcs_pair_count_static(lcs_t* h, double r_lo, double r_hi, int64_t* d_count)
{
    if (!h || !d_count || (reinterpret_cast<uintptr_t>(d_count) & 7u)) return LCS_ERR_INVALID_ARG;
    if (!(r_lo >= 0.0) || !(r_hi > r_lo) || !std::isfinite(r_hi)) return LCS_ERR_INVALID_ARG;
    const Geom& G = h->G;
    if (r_hi > G.L / 3.0) return LCS_ERR_INVALID_ARG;          // the cell list needs at least three cells per axis
    if (!h->have_particles || h->pushed) return LCS_ERR_STATE;
    if (h->sticky) return h->sticky;
    const size_t slots = (size_t)G.P * (size_t)G.cap;
    if (slots > (size_t)LCS_PAIR_COUNT_STATIC_MAX_SLOTS) return LCS_ERR_TOO_LARGE;
    int dev = -1;
    unsigned char* base = static_cast<unsigned char*>(pc_static_scratch(&dev));
    if (!base) return dev < 0 ? LCS_ERR_INVALID_ARG : LCS_ERR_CUDA;
    {   // the array of THIS device: the handle's particles must live on the device that is current
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, h->S.f[0]) != cudaSuccess) { cudaGetLastError(); return LCS_ERR_CUDA; }
        if (at.type == cudaMemoryTypeDevice && at.device != dev) return LCS_ERR_INVALID_ARG;
    }
    // carve: positions sorted by cell (three arrays of `slots` doubles), cell starts [ncell + 1], fill counters [ncell],
    // chunk sums of the scan [nchunks]
    const size_t arr_bytes = align_up(slots * 8);
    const size_t idx_bytes = 3 * arr_bytes;
    const size_t avail = (size_t)LCS_PAIR_COUNT_STATIC_BYTES - idx_bytes;     // >= 5 MiB by the slot limit
    const long long M = pair_cells_per_axis(G.L, r_hi, slots, avail);
    if (M < 3) return LCS_ERR_INVALID_ARG;
    const size_t ncell = (size_t)(M * M * M);
    const int nchunks = (int)((ncell + kScanChunk - 1) / kScanChunk);
    double* sx = reinterpret_cast<double*>(base);
    double* sy = reinterpret_cast<double*>(base + arr_bytes);
    double* sz = reinterpret_cast<double*>(base + 2 * arr_bytes);
    uint32_t* cellstart = reinterpret_cast<uint32_t*>(base + idx_bytes);
    uint32_t* cellfill = cellstart + ncell + 1;
    uint32_t* sums = cellfill + ncell;
    PairGeom Q;
    Q.M = (int)M; Q.inv_cell = (double)M / G.L; Q.L = G.L; Q.half_L = 0.5 * G.L; Q.lo2 = r_lo * r_lo; Q.hi2 = r_hi * r_hi;
    // the array still holds the last call's cell list: the counters and the result word must start at zero
    if (cudaMemsetAsync(cellstart, 0, (2 * ncell + 1) * 4, h->stream) != cudaSuccess ||
        cudaMemsetAsync(d_count, 0, 8, h->stream) != cudaSuccess) { cudaGetLastError(); return LCS_ERR_CUDA; }
    const dim3 pgrid((unsigned)((G.cap + 255) / 256), G.P);
    k_pc_count<<<pgrid, 256, 0, h->stream>>>(G, h->S, h->T, Q, cellstart);
    k_scan_sums<<<nchunks, 256, 0, h->stream>>>(cellstart, ncell, sums);
    k_scan_top<<<1, 1024, 0, h->stream>>>(sums, nchunks, cellstart + ncell);
    k_scan_apply<<<nchunks, 256, 0, h->stream>>>(cellstart, ncell, sums);
    k_pc_fill<<<pgrid, 256, 0, h->stream>>>(G, h->S, h->T, Q, cellstart, cellfill, sx, sy, sz);
    k_pc_pairs<<<(unsigned)((slots + 255) / 256), 256, 0, h->stream>>>(Q, cellstart, sx, sy, sz, cellstart + ncell,
                                                                        reinterpret_cast<unsigned long long*>(d_count));
    return check_launch(h, 6);
}
