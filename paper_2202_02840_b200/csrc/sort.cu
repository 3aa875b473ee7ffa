// sort.cu -- step a0 (first half): space-filling-curve keys, LSD radix sort, packed sorted state.
//
// PAPER.md:292 sorts particles into chaining-mesh bins and cuts RCB leaves of N_ppl particles; here the same
// locality is obtained by sorting on a 3b-bit Hilbert key (b <= 16 bits per axis, chosen from the smallest h) and cutting
// the sorted sequence into contiguous 32-particle leaves (tree.cu).  Every kernel here streams keys/payload once per pass.
#include "crk_internal.cuh"
#include <algorithm>
#include <mutex>
#include <stdarg.h>

namespace {

constexpr int SORT_THREADS = 256;
constexpr int SORT_ROUNDS = 8;                        // keys per lane (4 / 6 / 8 / 16 measured on 256^3: sort 1.23 / 1.11 / 1.14 / 1.35 ms)
constexpr int SORT_TILE = SORT_THREADS * SORT_ROUNDS; // 2048 keys per block
constexpr int SORT_WARPS = SORT_THREADS / 32;
constexpr int RADIX_BITS = 8;
constexpr int RADIX = 1 << RADIX_BITS;

// ---- 3-D Hilbert index (Skilling's transpose form), 16 bits per axis -> 48-bit key --------------------------
__device__ __forceinline__ uint64_t spread3(uint32_t v) {
    uint64_t x = v & 0x1fffffu;
    x = (x | x << 32) & 0x1f00000000ffffull;
    x = (x | x << 16) & 0x1f0000ff0000ffull;
    x = (x | x << 8) & 0x100f00f00f00f00full;
    x = (x | x << 4) & 0x10c30c30c30c30c3ull;
    x = (x | x << 2) & 0x1249249249249249ull;
    return x;
}

// b bits per axis -> 3 b-bit key (b <= 16)
__device__ __forceinline__ uint64_t hilbert_key(uint32_t X0, uint32_t X1, uint32_t X2, int b) {
    const uint32_t M = 1u << (b - 1);
    for (uint32_t Q = M; Q > 1; Q >>= 1) {
        const uint32_t P = Q - 1;
        // axis 0
        if (X0 & Q) X0 ^= P;
        // axis 1
        if (X1 & Q) X0 ^= P;
        else { uint32_t t = (X0 ^ X1) & P; X0 ^= t; X1 ^= t; }
        // axis 2
        if (X2 & Q) X0 ^= P;
        else { uint32_t t = (X0 ^ X2) & P; X0 ^= t; X2 ^= t; }
    }
    X1 ^= X0;
    X2 ^= X1;
    uint32_t t = 0;
    for (uint32_t Q = M; Q > 1; Q >>= 1)
        if (X2 & Q) t ^= Q - 1;
    X0 ^= t; X1 ^= t; X2 ^= t;
    return (spread3(X0) << 2) | (spread3(X1) << 1) | spread3(X2);
}

// smallest support radius of the set -> flag[1] (encoded so that a zero-initialised atomicMax finds the minimum); it
// decides how many key bits are worth computing and sorting (crk_sort_particles)
__global__ void __launch_bounds__(256) k_h_min(const float* __restrict__ h, int64_t n, int* __restrict__ flag) {
    uint32_t enc = 0u;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float hv = h[i];
        if (hv > 0.f && hv < 3.0e38f) enc = max(enc, 0x7f800000u - __float_as_uint(hv));
    }
    enc = __reduce_max_sync(0xffffffffu, enc);
    if ((threadIdx.x & 31) == 0 && enc != 0u) atomicMax((unsigned int*)flag + FW_HMIN, enc);
}

// validate (S13), key (Hilbert index of the 2^bits grid), and pack (x,y,z,h) so the later permutation gather
// moves 16-byte words
__global__ void __launch_bounds__(256) k_keys_pack(const float* __restrict__ x, const float* __restrict__ y,
                                                   const float* __restrict__ z, const float* __restrict__ h,
                                                   int64_t n, float L, int bits, uint64_t* __restrict__ keys,
                                                   uint32_t* __restrict__ vals, float4* __restrict__ posh_orig,
                                                   int* __restrict__ flag) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float xi = x[i], yi = y[i], zi = z[i], hi = h[i];
    const bool ok = (xi >= 0.f) && (xi < L) && (yi >= 0.f) && (yi < L) && (zi >= 0.f) && (zi < L) && (hi > 0.f) &&
                    (hi < 0.5f * L);
    if (!ok) atomicOr(flag, 1);
    const float s = (float)(1u << bits) / L;
    const uint32_t cmax = (1u << bits) - 1u;
    const uint32_t ix = min((uint32_t)fmaxf(xi * s, 0.f), cmax);
    const uint32_t iy = min((uint32_t)fmaxf(yi * s, 0.f), cmax);
    const uint32_t iz = min((uint32_t)fmaxf(zi * s, 0.f), cmax);
    keys[i] = hilbert_key(ix, iy, iz, bits);
    vals[i] = (uint32_t)i;
    posh_orig[i] = make_float4(xi, yi, zi, hi);
}

// per-tile digit histogram, stored digit-major so that one exclusive scan yields global stable offsets
__global__ void __launch_bounds__(SORT_THREADS) k_radix_hist(const uint64_t* __restrict__ keys, int64_t n, int shift,
                                                             uint32_t* __restrict__ hist, int nblk) {
    __shared__ uint32_t cnt[RADIX];
    cnt[threadIdx.x] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * SORT_TILE;
#pragma unroll
    for (int r = 0; r < SORT_ROUNDS; ++r) {
        const int64_t idx = base + r * SORT_THREADS + threadIdx.x;
        if (idx < n) atomicAdd(&cnt[(uint32_t)(keys[idx] >> shift) & (RADIX - 1)], 1u);
    }
    __syncthreads();
    hist[(int64_t)threadIdx.x * nblk + blockIdx.x] = cnt[threadIdx.x];
}

// stable scatter: each warp owns 256 consecutive keys (8 rounds of 32) and ranks them with match_any; the tile is then
// put in digit order in shared memory and written out as contiguous runs (one run per digit and CTA: ~8 keys = 64 B
// for uniform digits), so a warp store touches a handful of sectors instead of 32
struct ScatterSmem {
    uint64_t key[SORT_TILE];                 // tile in local digit order
    uint32_t val[SORT_TILE];
    uint32_t wcnt[SORT_WARPS][RADIX];        // per-warp digit counts -> per-warp base inside the digit run
    uint32_t lbase[RADIX];                   // first local position of the digit run
    uint32_t gbase[RADIX];                   // first global position of the digit run
    uint32_t wsum[SORT_WARPS];
};
__global__ void __launch_bounds__(SORT_THREADS) k_radix_scatter(const uint64_t* __restrict__ keys_in,
                                                                const uint32_t* __restrict__ vals_in,
                                                                uint64_t* __restrict__ keys_out,
                                                                uint32_t* __restrict__ vals_out, int64_t n, int shift,
                                                                const uint32_t* __restrict__ offs, int nblk) {
    extern __shared__ __align__(16) unsigned char scatter_raw[];
    ScatterSmem& S = *(ScatterSmem*)scatter_raw;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int q = threadIdx.x; q < SORT_WARPS * RADIX; q += SORT_THREADS) (&S.wcnt[0][0])[q] = 0;
    __syncthreads();
    const int64_t tbase = (int64_t)blockIdx.x * SORT_TILE;
    const int64_t wbase = tbase + (int64_t)w * (32 * SORT_ROUNDS);
    uint64_t k[SORT_ROUNDS];
    uint32_t v[SORT_ROUNDS];
    uint32_t rk[SORT_ROUNDS];     // first: digit | rank among equal digits of the round << 9 | group size << 15 ; then: rank in (warp, digit)
    const uint32_t lt = (1u << lane) - 1u;
    // phase 1 (independent per round, so the loads and the match instructions overlap): digit, rank within the round
#pragma unroll
    for (int r = 0; r < SORT_ROUNDS; ++r) {
        const int64_t idx = wbase + r * 32 + lane;
        const bool valid = idx < n;
        k[r] = valid ? keys_in[idx] : 0ull;
        v[r] = valid ? vals_in[idx] : 0u;
    }
#pragma unroll
    for (int r = 0; r < SORT_ROUNDS; ++r) {
        const bool valid = (wbase + r * 32 + lane) < n;
        const uint32_t d = valid ? ((uint32_t)(k[r] >> shift) & (RADIX - 1)) : (uint32_t)RADIX;
        const uint32_t peers = __match_any_sync(0xffffffffu, d);
        rk[r] = d | ((uint32_t)__popc(peers & lt) << 9) | ((uint32_t)__popc(peers) << 15);
    }
    // phase 2 (serial over rounds: stable counts per warp and digit)
#pragma unroll
    for (int r = 0; r < SORT_ROUNDS; ++r) {
        const uint32_t d = rk[r] & 0x1ffu, rank = (rk[r] >> 9) & 0x3fu, gsz = rk[r] >> 15;
        const bool valid = d < (uint32_t)RADIX;
        uint32_t prev = 0;
        if (valid) prev = S.wcnt[w][d];
        __syncwarp();
        if (valid && rank == 0) S.wcnt[w][d] = prev + gsz;
        __syncwarp();
        rk[r] = prev + rank;
    }
    __syncthreads();
    // phase 3: thread d owns digit d (256 threads <-> 256 digits): per-warp bases inside the run, run length, block scan
    {
        const int d = threadIdx.x;
        uint32_t run = 0;
#pragma unroll
        for (int ww = 0; ww < SORT_WARPS; ++ww) {
            const uint32_t cc = S.wcnt[ww][d];
            S.wcnt[ww][d] = run;
            run += cc;
        }
        // exclusive scan of the 256 run lengths
        uint32_t inc = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) S.wsum[w] = inc;
        __syncthreads();
        uint32_t wpre = 0;
#pragma unroll
        for (int ww = 0; ww < SORT_WARPS; ++ww) wpre += (ww < w) ? S.wsum[ww] : 0u;
        S.lbase[d] = wpre + inc - run;
        S.gbase[d] = offs[(int64_t)d * nblk + blockIdx.x];
    }
    __syncthreads();
    // phase 4: tile -> shared memory in digit order
#pragma unroll
    for (int r = 0; r < SORT_ROUNDS; ++r) {
        const int64_t idx = wbase + r * 32 + lane;
        if (idx < n) {
            const uint32_t d = (uint32_t)(k[r] >> shift) & (RADIX - 1);
            const uint32_t lp = S.lbase[d] + S.wcnt[w][d] + rk[r];
            S.key[lp] = k[r];
            S.val[lp] = v[r];
        }
    }
    __syncthreads();
    // phase 5: contiguous runs out
    const int cnt = (int)min((int64_t)SORT_TILE, n - tbase);
    for (int p = threadIdx.x; p < cnt; p += SORT_THREADS) {
        const uint64_t kk = S.key[p];
        const uint32_t d = (uint32_t)(kk >> shift) & (RADIX - 1);
        const uint32_t pos = S.gbase[d] + ((uint32_t)p - S.lbase[d]);
        keys_out[pos] = kk;
        vals_out[pos] = S.val[p];
    }
}

// ---- exclusive scan (u32), out has n+1 entries, out[n] = total ------------------------------------------------
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_block(const uint32_t* __restrict__ in, uint32_t* __restrict__ out,
                                                             int64_t n_in, int64_t n_out, uint32_t* __restrict__ sums) {
    __shared__ uint32_t wsum[SCAN_THREADS / 32];
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    uint32_t v[SCAN_ITEMS];
    uint32_t tot = 0;
#pragma unroll
    for (int q = 0; q < SCAN_ITEMS; ++q) {
        const int64_t i = base + q;
        v[q] = (i < n_in) ? in[i] : 0u;
        tot += v[q];
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t inc = tot;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    uint32_t woff = 0;
    for (int q = 0; q < w; ++q) woff += wsum[q];
    uint32_t run = woff + inc - tot;
#pragma unroll
    for (int q = 0; q < SCAN_ITEMS; ++q) {
        const int64_t i = base + q;
        if (i < n_out) out[i] = run;
        run += v[q];
    }
    if (threadIdx.x == SCAN_THREADS - 1 && sums) sums[blockIdx.x] = woff + inc;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_add(uint32_t* __restrict__ out, int64_t n_out,
                                                           const uint32_t* __restrict__ sums_scanned) {
    const uint32_t add = sums_scanned[blockIdx.x];
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE;
    for (int q = threadIdx.x; q < SCAN_TILE; q += SCAN_THREADS) {
        const int64_t i = base + q;
        if (i < n_out) out[i] += add;
    }
}

int scan_rec(crk_ctx* c, const uint32_t* in, uint32_t* out, int64_t n_in, int64_t n_out, uint32_t* tmp) {
    const int64_t nblk = (n_out + SCAN_TILE - 1) / SCAN_TILE;
    if (nblk <= 1) {
        k_scan_block<<<1, SCAN_THREADS, 0, c->stream>>>(in, out, n_in, n_out, nullptr);
        return crk_check_launch(c, "k_scan_block");
    }
    uint32_t* sums = tmp;
    uint32_t* sums_scanned = tmp + nblk;                 // nblk + 1 entries
    k_scan_block<<<(unsigned)nblk, SCAN_THREADS, 0, c->stream>>>(in, out, n_in, n_out, sums);
    CRK_TRY(crk_check_launch(c, "k_scan_block"));
    CRK_TRY(scan_rec(c, sums, sums_scanned, nblk, nblk + 1, sums_scanned + nblk + 1));
    k_scan_add<<<(unsigned)nblk, SCAN_THREADS, 0, c->stream>>>(out, n_out, sums_scanned);
    return crk_check_launch(c, "k_scan_add");
}

// sorted (x,y,z,h) by a 16-byte gather through the permutation, and the leaf bounding boxes in the same pass
__global__ void __launch_bounds__(256) k_gather_leaves(const float4* __restrict__ posh_orig,
                                                       const uint32_t* __restrict__ perm, int64_t n, int64_t nl,
                                                       float4* __restrict__ posh, float4* __restrict__ leaf_lo,
                                                       float4* __restrict__ leaf_hi) {
    const int lane = threadIdx.x & 31;
    const int64_t leaf = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (leaf >= nl) return;
    const int64_t k = leaf * CRK_LEAF + lane;
    const float inf = __int_as_float(0x7f800000);
    float4 lo = make_float4(inf, inf, inf, 0.f), hi = make_float4(-inf, -inf, -inf, inf);
    if (k < n) {
        const float4 p = posh_orig[perm[k]];
        posh[k] = p;
        lo = make_float4(p.x, p.y, p.z, p.w);
        hi = make_float4(p.x, p.y, p.z, p.w);
    } else {
        posh[k] = make_float4(3.0e30f, 3.0e30f, 3.0e30f, 0.0f);   // padding lanes of the last leaf: never a neighbour
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        lo.x = fminf(lo.x, __shfl_xor_sync(0xffffffffu, lo.x, o));
        lo.y = fminf(lo.y, __shfl_xor_sync(0xffffffffu, lo.y, o));
        lo.z = fminf(lo.z, __shfl_xor_sync(0xffffffffu, lo.z, o));
        lo.w = fmaxf(lo.w, __shfl_xor_sync(0xffffffffu, lo.w, o));   // hmax
        hi.x = fmaxf(hi.x, __shfl_xor_sync(0xffffffffu, hi.x, o));
        hi.y = fmaxf(hi.y, __shfl_xor_sync(0xffffffffu, hi.y, o));
        hi.z = fmaxf(hi.z, __shfl_xor_sync(0xffffffffu, hi.z, o));
        hi.w = fminf(hi.w, __shfl_xor_sync(0xffffffffu, hi.w, o));   // hmin
    }
    if (lane == 0) {
        leaf_lo[leaf] = lo;
        leaf_hi[leaf] = hi;
    }
}

}  // namespace

int crk_exclusive_scan_u32(crk_ctx* c, const uint32_t* in, uint32_t* out, int64_t n, DevBuf& tmp) {
    // scratch: sum over levels of (2*nblk + 2)
    size_t need = 0;
    for (int64_t m = n + 1; m > 1;) {
        const int64_t nblk = (m + SCAN_TILE - 1) / SCAN_TILE;
        need += (size_t)(2 * nblk + 2);
        if (nblk <= 1) break;
        m = nblk + 1;
    }
    CRK_TRY(crk_ensure(c, tmp, need * sizeof(uint32_t) + 64));
    return scan_rec(c, in, out, n, n + 1, (uint32_t*)tmp.p);
}

// Key bits worth sorting: cells of half the smallest support radius order everything the leaves need (a finer order inside
// such a cell does not make a 32-particle leaf more compact than its h).  The top 3 b bits of a Hilbert key are the key of
// the b-bit grid, so only b levels of the curve are computed and sorted.
int crk_key_bits_from_hmin(const crk_ctx* c, uint32_t enc) {
    int bits = CRK_KEY_BITS;
    if (enc != 0u) {
        const uint32_t hb = 0x7f800000u - enc;
        float hmin;
        memcpy(&hmin, &hb, sizeof(hmin));
        if (hmin > 0.f) {
            const double cells = 2.0 * (double)c->prm.box / (double)hmin;
            bits = 1;
            while (bits < CRK_KEY_BITS && (double)(1u << bits) < cells) ++bits;
        }
    }
    return bits < 6 ? 6 : bits;
}

// smallest h of the set -> status word FW_HMIN (read back with the other status words at the end of the build); sync = true:
// read it now (first build of a context, when no key width is known yet)
int crk_measure_hmin(crk_ctx* c, const float* h, bool sync, uint32_t* enc_out) {
    k_h_min<<<(unsigned)std::min<int64_t>((c->n + 255) / 256, 1184), 256, 0, c->stream>>>(h, c->n, (int*)c->flag.p);
    CRK_TRY(crk_check_launch(c, "k_h_min"));
    if (sync) {
        CRK_CUDA(c, cudaMemcpyAsync(c->h_flag + FW_HMIN, (int*)c->flag.p + FW_HMIN, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
        CRK_CUDA(c, cudaStreamSynchronize(c->stream));
        *enc_out = (uint32_t)c->h_flag[FW_HMIN];
    }
    return CRK_OK;
}

int crk_sort_particles(crk_ctx* c, const float* x, const float* y, const float* z, const float* h, int bits) {
    const int64_t n = c->n;
    const int64_t nl = c->nl;
    for (int q = 0; q < 2; ++q) {
        CRK_TRY(crk_ensure(c, c->keys[q], (size_t)n * sizeof(uint64_t)));
        CRK_TRY(crk_ensure(c, c->vals[q], (size_t)n * sizeof(uint32_t)));
    }
    CRK_TRY(crk_ensure(c, c->posh_orig, (size_t)n * sizeof(float4)));
    CRK_TRY(crk_ensure(c, c->posh, (size_t)nl * CRK_LEAF * sizeof(float4)));
    const int nblk = (int)((n + SORT_TILE - 1) / SORT_TILE);
    CRK_TRY(crk_ensure(c, c->hist, ((size_t)RADIX * nblk + 1) * 2 * sizeof(uint32_t)));
    uint32_t* hist = (uint32_t*)c->hist.p;
    uint32_t* offs = hist + (size_t)RADIX * nblk + 1;
    k_keys_pack<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(x, y, z, h, n, c->prm.box, bits, (uint64_t*)c->keys[0].p,
                                                                    (uint32_t*)c->vals[0].p, (float4*)c->posh_orig.p,
                                                                    (int*)c->flag.p);
    CRK_TRY(crk_check_launch(c, "k_keys_pack"));
    CRK_CUDA(c, cudaFuncSetAttribute(k_radix_scatter, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(ScatterSmem)));
    int cur = 0;
    c->st.sort_passes = (3 * bits + RADIX_BITS - 1) / RADIX_BITS;
    for (int shift = 0; shift < 3 * bits; shift += RADIX_BITS) {
        k_radix_hist<<<nblk, SORT_THREADS, 0, c->stream>>>((const uint64_t*)c->keys[cur].p, n, shift, hist, nblk);
        CRK_TRY(crk_check_launch(c, "k_radix_hist"));
        CRK_TRY(crk_exclusive_scan_u32(c, hist, offs, (int64_t)RADIX * nblk, c->scan_tmp));
        k_radix_scatter<<<nblk, SORT_THREADS, sizeof(ScatterSmem), c->stream>>>((const uint64_t*)c->keys[cur].p,
                                                              (const uint32_t*)c->vals[cur].p,
                                                              (uint64_t*)c->keys[cur ^ 1].p,
                                                              (uint32_t*)c->vals[cur ^ 1].p, n, shift, offs, nblk);
        CRK_TRY(crk_check_launch(c, "k_radix_scatter"));
        cur ^= 1;
    }
    c->perm = (int32_t*)c->vals[cur].p;

    // leaves (level 0 of the tree) are written by the gather; tree.cu sizes the node arrays
    int64_t total = 0, cnt = nl;
    int lev = 0;
    while (true) {
        c->level_off[lev] = total;
        c->level_cnt[lev] = cnt;
        total += cnt;
        if (cnt <= CRK_BVH_FAN || lev + 1 >= CRK_MAX_LEVELS) break;
        cnt = (cnt + CRK_BVH_FAN - 1) / CRK_BVH_FAN;
        ++lev;
    }
    c->n_levels = lev + 1;
    CRK_TRY(crk_ensure(c, c->leaf_lo, (size_t)total * sizeof(float4)));
    CRK_TRY(crk_ensure(c, c->leaf_hi, (size_t)total * sizeof(float4)));
    const int wpb = 8;
    k_gather_leaves<<<(unsigned)((nl + wpb - 1) / wpb), wpb * 32, 0, c->stream>>>(
        (const float4*)c->posh_orig.p, (const uint32_t*)c->perm, n, nl, (float4*)c->posh.p, (float4*)c->leaf_lo.p,
        (float4*)c->leaf_hi.p);
    return crk_check_launch(c, "k_gather_leaves");
}

// ---- crk_sfc_order_noalloc (include/crk.h): the sort above for callers that must not allocate --------------------------
// Hosts that hand the whole device to their own arena at start-up, or that cannot take the device-wide stall of a
// cudaMalloc in the middle of a time step, get the curve order from here: same kernels, same launch order as
// crk_measure_hmin + crk_sort_particles, but every buffer the sort needs is a slice of ONE array that is part of the
// library's device image.  Nothing below calls cudaMalloc, cudaFree, cudaMallocHost or anything that does.
namespace {

constexpr size_t na_al(size_t b) { return (b + 255) & ~(size_t)255; }
constexpr size_t NA_N = CRK_NOALLOC_MAX_N;
constexpr size_t NA_NBLK = (NA_N + SORT_TILE - 1) / SORT_TILE;
constexpr size_t NA_HIST_WORDS = (size_t)RADIX * NA_NBLK + 1;      // digit-major histogram; its scan has one entry more
constexpr size_t NA_SCAN_WORDS = 4096;                             // block sums of the scan (40 words at the maximal n)
constexpr size_t NA_OFF_FLAG = 0;                                  // FW_WORDS status words; FW_ERROR and FW_HMIN are used
constexpr size_t NA_OFF_KEYS0 = NA_OFF_FLAG + na_al(FW_WORDS * sizeof(int));
constexpr size_t NA_OFF_KEYS1 = NA_OFF_KEYS0 + na_al(NA_N * sizeof(uint64_t));
constexpr size_t NA_OFF_VALS0 = NA_OFF_KEYS1 + na_al(NA_N * sizeof(uint64_t));
constexpr size_t NA_OFF_VALS1 = NA_OFF_VALS0 + na_al(NA_N * sizeof(uint32_t));
constexpr size_t NA_OFF_POSH = NA_OFF_VALS1 + na_al(NA_N * sizeof(uint32_t));
constexpr size_t NA_OFF_HIST = NA_OFF_POSH + na_al(NA_N * sizeof(float4));
constexpr size_t NA_OFF_OFFS = NA_OFF_HIST + na_al(NA_HIST_WORDS * sizeof(uint32_t));
constexpr size_t NA_OFF_SCAN = NA_OFF_OFFS + na_al(NA_HIST_WORDS * sizeof(uint32_t));
constexpr size_t NA_BYTES = NA_OFF_SCAN + na_al(NA_SCAN_WORDS * sizeof(uint32_t));
static_assert(NA_BYTES == CRK_NOALLOC_SCRATCH_BYTES, "include/crk.h states the size of the fixed scratch array");

// The scratch itself.  In HOST code this name is only a handle for the runtime's symbol calls -- it is not a device
// address, and a kernel handed `na_scratch` directly would fault (or, on a system where the GPU can reach host memory,
// quietly work on the wrong bytes).  Host code therefore asks cudaGetSymbolAddress for the device's copy, once per device.
static __device__ __align__(256) unsigned char na_scratch[NA_BYTES];

constexpr int NA_MAX_DEVICES = 64;
unsigned char* na_dev_ptr[NA_MAX_DEVICES] = {};   // device address of na_scratch on device d, 0 = not looked up yet
std::mutex na_mu;                                  // guards na_dev_ptr (set-up only; it does not serialise the GPU work)

int na_fail(char* errbuf, int errbuf_len, int code, const char* fmt, ...) {
    if (errbuf && errbuf_len > 0) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(errbuf, (size_t)errbuf_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// device address of the scratch array on the CURRENT device; looked up on the first call made with that device current
int na_scratch_for_current_device(unsigned char** out, char* errbuf, int errbuf_len) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return na_fail(errbuf, errbuf_len, CRK_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= NA_MAX_DEVICES)
        return na_fail(errbuf, errbuf_len, CRK_ECUDA, "crk_sfc_order_noalloc: device ordinal %d is beyond the %d this entry point keeps track of", dev, NA_MAX_DEVICES);
    std::lock_guard<std::mutex> lock(na_mu);
    if (!na_dev_ptr[dev]) {
        unsigned char* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, na_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return na_fail(errbuf, errbuf_len, CRK_ECUDA, "cudaGetSymbolAddress(fixed scratch array) on device %d: %s", dev, cudaGetErrorString(e));
        }
        na_dev_ptr[dev] = p;
    }
    *out = na_dev_ptr[dev];
    return CRK_OK;
}

#define NA_CUDA(call)                                                                                                   \
    do {                                                                                                                \
        cudaError_t e__ = (call);                                                                                       \
        if (e__ != cudaSuccess) return na_fail(errbuf, errbuf_len, CRK_ECUDA, "crk_sfc_order_noalloc: %s: %s", #call, cudaGetErrorString(e__)); \
    } while (0)

}  // namespace

extern "C" int crk_sfc_order_noalloc(void* cuda_stream, int64_t n, const float* x, const float* y, const float* z, const float* h,
                                     float box, int32_t* perm, char* errbuf, int errbuf_len) {
    if (errbuf && errbuf_len > 0) errbuf[0] = 0;
    if (n < 0) return na_fail(errbuf, errbuf_len, CRK_EINVAL, "crk_sfc_order_noalloc: n = %lld is negative", (long long)n);
    if (n > (int64_t)NA_N)
        return na_fail(errbuf, errbuf_len, CRK_EINVAL,
                       "crk_sfc_order_noalloc: n = %lld exceeds CRK_NOALLOC_MAX_N = %lld, the capacity of the fixed scratch array; "
                       "use crk_build_cells + crk_get_perm (which allocate) for larger sets",
                       (long long)n, (long long)NA_N);
    if (!(box > 0.f)) return na_fail(errbuf, errbuf_len, CRK_EINVAL, "crk_sfc_order_noalloc: box must be positive");
    if (n > 0 && (!x || !y || !z || !h || !perm)) return na_fail(errbuf, errbuf_len, CRK_EINVAL, "crk_sfc_order_noalloc: null pointer");
    // set-up of this device (first call only): also with n = 0, so that a start-up call outside any capture does it
    unsigned char* S = nullptr;
    CRK_TRY(na_scratch_for_current_device(&S, errbuf, errbuf_len));
    if (n == 0) return CRK_OK;

    cudaStream_t st = (cudaStream_t)cuda_stream;
    int* flag = (int*)(S + NA_OFF_FLAG);
    uint64_t* keys[2] = {(uint64_t*)(S + NA_OFF_KEYS0), (uint64_t*)(S + NA_OFF_KEYS1)};
    uint32_t* vals[2] = {(uint32_t*)(S + NA_OFF_VALS0), (uint32_t*)(S + NA_OFF_VALS1)};
    float4* posh_orig = (float4*)(S + NA_OFF_POSH);
    uint32_t* hist = (uint32_t*)(S + NA_OFF_HIST);
    uint32_t* offs = (uint32_t*)(S + NA_OFF_OFFS);
    uint32_t* scan_tmp = (uint32_t*)(S + NA_OFF_SCAN);

    // launch bookkeeping of the helpers above goes through a context object; this one lives on the host stack, owns nothing
    // and is never passed to anything that allocates
    crk_ctx tmp;
    tmp.stream = st;
    tmp.prm.box = box;
    tmp.n = n;
    tmp.err[0] = 0;

    // the array keeps what the last call left in it: the two status words (range flag, encoded smallest h) must start at zero
    NA_CUDA(cudaMemsetAsync(flag, 0, FW_WORDS * sizeof(int), st));
    k_h_min<<<(unsigned)std::min<int64_t>((n + 255) / 256, 1184), 256, 0, st>>>(h, n, flag);
    NA_CUDA(cudaGetLastError());
    int enc_host = 0;
    NA_CUDA(cudaMemcpyAsync(&enc_host, flag + FW_HMIN, sizeof(int), cudaMemcpyDeviceToHost, st));
    NA_CUDA(cudaStreamSynchronize(st));
    const int bits = crk_key_bits_from_hmin(&tmp, (uint32_t)enc_host);     // as the first crk_build_cells of a context

    const int nblk = (int)((n + SORT_TILE - 1) / SORT_TILE);
    {   // block sums of the scan must fit their slice (they do for every n <= CRK_NOALLOC_MAX_N; checked, not assumed)
        size_t need = 0;
        for (int64_t m = (int64_t)RADIX * nblk + 1; m > 1;) {
            const int64_t nb = (m + SCAN_TILE - 1) / SCAN_TILE;
            need += (size_t)(2 * nb + 2);
            if (nb <= 1) break;
            m = nb + 1;
        }
        if (need > NA_SCAN_WORDS || (size_t)RADIX * nblk + 1 > NA_HIST_WORDS)
            return na_fail(errbuf, errbuf_len, CRK_EINVAL, "crk_sfc_order_noalloc: n = %lld does not fit the fixed scratch array", (long long)n);
    }
    k_keys_pack<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(x, y, z, h, n, box, bits, keys[0], vals[0], posh_orig, flag);
    NA_CUDA(cudaGetLastError());
    NA_CUDA(cudaFuncSetAttribute(k_radix_scatter, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(ScatterSmem)));
    int cur = 0;
    for (int shift = 0; shift < 3 * bits; shift += RADIX_BITS) {
        k_radix_hist<<<nblk, SORT_THREADS, 0, st>>>(keys[cur], n, shift, hist, nblk);      // writes every entry it owns: no clearing
        NA_CUDA(cudaGetLastError());
        if (scan_rec(&tmp, hist, offs, (int64_t)RADIX * nblk, (int64_t)RADIX * nblk + 1, scan_tmp) != CRK_OK)
            return na_fail(errbuf, errbuf_len, CRK_ECUDA, "crk_sfc_order_noalloc: %s", tmp.err);
        k_radix_scatter<<<nblk, SORT_THREADS, sizeof(ScatterSmem), st>>>(keys[cur], vals[cur], keys[cur ^ 1], vals[cur ^ 1], n, shift,
                                                                         offs, nblk);
        NA_CUDA(cudaGetLastError());
        cur ^= 1;
    }
    NA_CUDA(cudaMemcpyAsync(perm, vals[cur], (size_t)n * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
    int err_host = 0;
    NA_CUDA(cudaMemcpyAsync(&err_host, flag + FW_ERROR, sizeof(int), cudaMemcpyDeviceToHost, st));
    NA_CUDA(cudaStreamSynchronize(st));
    if (err_host & 1)
        return na_fail(errbuf, errbuf_len, CRK_ERANGE, "input out of range: need 0 <= x,y,z < box and 0 < h < box/2");
    return CRK_OK;
}
