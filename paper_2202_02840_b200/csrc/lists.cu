// lists.cu -- step a0 (third part): per-particle neighbour lists, built once per crk_build_cells and reused by all
// pair sweeps ("all hydro operators utilize the same interaction list, which need only be assembled once per hydro
// subcycle, and reused for each kernel", PAPER.md:302 -- here taken down to particle pairs).
//
// One warp = one 32-particle leaf, one lane = one particle i.  For every neighbour leaf of the leaf interaction list
// (tree.cu) lane l takes particle l of that leaf and culls it against the query leaf's box; survivors go to a small tile;
// every staged j is then tested against every lane's i with the prescribed FP32 predicate (S3), two candidates
// per instruction stream with the packed FP32 forms of sm_100 (add/mul/fma.rn.f32x2: each half is rounded to nearest, so
// the bits are those of the scalar sequence).  A candidate accepted by at least one lane receives the next candidate
// index c of the current segment; lane i appends c to its entries, flagged "symmetric only" when h_i^2 <= r2 < h_j^2
// (a pair of Eqs. 17-18 that is not in the gather set of Eqs. 13-14).  A segment is written to the arena as
// header | cand[C] | ell[K][32]  (layout in crk_internal.cuh); it is cut when the candidate or entry capacity would
// overflow, so leaves in strongly clustered regions own a chain of segments.
#include "crk_internal.cuh"

namespace {

constexpr int LW = 2;   // warps (= leaves) per CTA

struct ListArgs {
    int64_t n, nl;
    float L, half;
    const uint32_t* __restrict__ cnt;      // entries of each leaf's interaction list
    const uint32_t* __restrict__ list;     // leaf q owns list[q * cap ...]
    uint32_t cap;
    const float4* __restrict__ posh;
    const float4* __restrict__ leaf_lo;
    const float4* __restrict__ leaf_hi;
    uint4* arena;
    unsigned long long arena_cap;          // units
    unsigned long long* counter;           // next free unit (unit 0 is reserved as "none")
    uint4* __restrict__ seg_first;         // dense copy of each leaf's first header (.w = its arena unit)
    uint16_t* __restrict__ leaf_cnt;       // [nl][32]
    uint32_t* __restrict__ cand_first;     // [nl][CRK_CAND_STRIDE] candidates of each leaf's first segment
    int* flag;                             // status words (CRK_CHECKED builds write FW_CHECK)
};

struct WarpSmem {
    float4 ta[(CRK_TCULL + 2) / 2];   // candidates 2t, 2t+1: (-x_a, -x_b, -y_a, -y_b)
    float4 tb[(CRK_TCULL + 2) / 2];   //                      (-z_a, -z_b, h_a^2, h_b^2)
    __align__(8) uint32_t tidx[CRK_TCULL + 2];
    uint32_t cand[CRK_CCAP];
    __align__(16) uint16_t queue[CRK_QCAP][32];   // same layout as a segment's entry block: emit copies it in 16-byte units
};

// lower bound of |wrap(x_i - x_j)| on one axis for x_i in [lo,hi] (monotone float ops, so nothing is lost)
__device__ __forceinline__ float gap1(float lo, float hi, float x) {
    return fmaxf(0.f, fmaxf(__fsub_rn(lo, x), __fsub_rn(x, hi)));
}
__device__ __forceinline__ float gap1_wrap(float lo, float hi, float x, float L) {
    const float dmin = __fsub_rn(lo, x), dmax = __fsub_rn(hi, x);
    const float g0 = fmaxf(0.f, fmaxf(dmin, -dmax));
    const float gp = fmaxf(0.f, fmaxf(__fsub_rn(L, dmax), __fsub_rn(dmin, L)));
    const float gm = fmaxf(0.f, fmaxf(__fadd_rn(dmin, L), __fsub_rn(-L, dmax)));
    return fminf(g0, fminf(gp, gm));
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void sts_u16_if(uint32_t addr, uint32_t v, bool pred) {
    asm volatile("{ .reg .pred p; setp.ne.b32 p, %2, 0; @p st.shared.u16 [%0], %1; }" ::"r"(addr), "h"((uint16_t)v), "r"((int)pred) : "memory");
}
// minimum-image wrap of both halves (S3: d > L/2 -> d - L, d < -L/2 -> d + L); adding 0 leaves the other values untouched
__device__ __forceinline__ float2 wrap2(float2 d, float L, float half, bool& wa, bool& wb) {
    const float sa = d.x > half ? -L : (d.x < -half ? L : 0.f);
    const float sb = d.y > half ? -L : (d.y < -half ? L : 0.f);
    wa = wa || (sa != 0.f);
    wb = wb || (sb != 0.f);
    return __fadd2_rn(d, make_float2(sa, sb));
}

// test every staged candidate against the lane's particle; returns the new candidate count of the segment.
// Branch-free, two candidates per trip (the tile is padded to an even count with a far-away sentinel): about 3 of 4
// culled candidates are accepted by some lane, so predicated appends beat a vote-and-branch per candidate.  A candidate
// accepted by at least one lane receives the next slot of the segment (kept = bit mask of those candidates; their indices
// are compacted into S.cand after the loop); keeping every culled candidate instead was measured: a third more slots, half of
// the leaves spill into a second segment and every sweep stages and pays for them (forces 11.0 -> 12.8 ms).
// SELF: the tile holds the query leaf itself in lane order (C = 0), so j = i is the candidate t = lane, and every candidate
// keeps its slot.
template <bool WRAP, bool SELF>
__device__ __forceinline__ int test_tile(WarpSmem& S, int* flag, int fill, int C, int& g, bool& wflag, int lane,
                                         float xi, float yi, float zi, float hi2, float L, float half) {
    uint32_t gp = smem_u32(&S.queue[g][lane]);                  // next entry of this lane (row stride 64 bytes)
    const float2 xi2 = make_float2(xi, xi), yi2 = make_float2(yi, yi), zi2 = make_float2(zi, zi);
    const int C0 = C;
    uint32_t kept = 0u, bit = 1u, Cu = (uint32_t)C, Cs = (uint32_t)C | CRK_ELL_SYM;
    for (int t0 = 0; t0 < fill; t0 += 2) {
        const float4 pa = S.ta[t0 >> 1], pb = S.tb[t0 >> 1];
        float2 dx = __fadd2_rn(xi2, make_float2(pa.x, pa.y));    // x_i - x_j (the tile holds -x_j)
        float2 dy = __fadd2_rn(yi2, make_float2(pa.z, pa.w));
        float2 dz = __fadd2_rn(zi2, make_float2(pb.x, pb.y));
        bool wr[2] = {false, false};
        if (WRAP) {
            dx = wrap2(dx, L, half, wr[0], wr[1]);
            dy = wrap2(dy, L, half, wr[0], wr[1]);
            dz = wrap2(dz, L, half, wr[0], wr[1]);
        }
        const float2 r2v = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __fmul2_rn(dx, dx)));
        const float r2[2] = {r2v.x, r2v.y}, hj2[2] = {pb.z, pb.w};
        if (!SELF) {
            // one candidate = ten instructions, written out because the compiler turns the conditional increments into add + move
            // pairs and rebuilds the bit of `kept` with a shift, a select and an or: two compares, the acceptance vote, the
            // entry word, one predicated 16-bit store, and four predicated updates (queue pointer, kept mask, C, C | SYM)
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                if (WRAP) {
                    uint32_t hit;
                    asm volatile(
                        "{\n"
                        ".reg .pred pg, ps, pa;\n"
                        ".reg .b32 e;\n"
                        ".reg .b16 eh;\n"
                        "setp.lt.f32 pg, %6, %7;\n"                    // gather: r2 < h_i^2 (Eqs. 13-14)
                        "setp.lt.or.f32 ps, %6, %8, pg;\n"             // symmetric: r2 < max(h_i^2, h_j^2) (Eqs. 17-18)
                        "vote.sync.any.pred pa, ps, 0xffffffff;\n"     // a candidate accepted by some lane gets the next slot
                        "selp.b32 e, %2, %3, pg;\n"
                        "or.b32 e, e, %9;\n"                           // CRK_ELL_WRAP: the pair crosses the periodic boundary
                        "cvt.u16.u32 eh, e;\n"
                        "@ps st.shared.u16 [%0], eh;\n"
                        "@ps add.u32 %0, %0, 64;\n"
                        "selp.u32 %5, 1, 0, ps;\n"
                        "@pa or.b32 %1, %1, %4;\n"
                        "@pa add.u32 %2, %2, 1;\n"
                        "@pa add.u32 %3, %3, 1;\n"
                        "shl.b32 %4, %4, 1;\n"
                        "}"
                        : "+r"(gp), "+r"(kept), "+r"(Cu), "+r"(Cs), "+r"(bit), "=r"(hit)
                        : "f"(r2[u]), "f"(hi2), "f"(hj2[u]), "r"(wr[u] ? CRK_ELL_WRAP : 0u)
                        : "memory");
                    wflag = wflag || (wr[u] && hit != 0u);
                } else {
                    asm volatile(
                        "{\n"
                        ".reg .pred pg, ps, pa;\n"
                        ".reg .b32 e;\n"
                        ".reg .b16 eh;\n"
                        "setp.lt.f32 pg, %5, %6;\n"
                        "setp.lt.or.f32 ps, %5, %7, pg;\n"
                        "vote.sync.any.pred pa, ps, 0xffffffff;\n"
                        "selp.b32 e, %2, %3, pg;\n"
                        "cvt.u16.u32 eh, e;\n"
                        "@ps st.shared.u16 [%0], eh;\n"
                        "@ps add.u32 %0, %0, 64;\n"
                        "@pa or.b32 %1, %1, %4;\n"
                        "@pa add.u32 %2, %2, 1;\n"
                        "@pa add.u32 %3, %3, 1;\n"
                        "shl.b32 %4, %4, 1;\n"
                        "}"
                        : "+r"(gp), "+r"(kept), "+r"(Cu), "+r"(Cs), "+r"(bit)
                        : "f"(r2[u]), "f"(hi2), "f"(hj2[u])
                        : "memory");
                }
                CRK_CHECK(flag, gp <= smem_u32(&S.queue[CRK_QCAP - 1][31]) + 66u, 0);          // entry queue row < CRK_QCAP
                CRK_CHECK(flag, Cu <= (uint32_t)CRK_CCAP, 1);                                    // candidate slot < CRK_CCAP
            }
        } else {
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                bool ag = r2[u] < hi2;                                         // gather: Eqs. 13-14
                bool as = ag || (r2[u] < hj2[u]);                              // symmetric: r2 < max(h_i^2, h_j^2), Eqs. 17-18
                const bool notself = (t0 + u) != lane;                         // the tile is the leaf itself in lane order
                ag = ag && notself;
                as = as && notself;
                uint32_t e = ag ? Cu : Cs;
                if (WRAP) {
                    e |= wr[u] ? CRK_ELL_WRAP : 0u;
                    wflag = wflag || (wr[u] && as);
                }
                CRK_CHECK(flag, !as || gp < smem_u32(&S.queue[CRK_QCAP - 1][31]) + 2u, 0);   // entry queue row < CRK_QCAP
                CRK_CHECK(flag, Cu < (uint32_t)CRK_CCAP, 1);                                   // candidate slot < CRK_CCAP
                sts_u16_if(gp, e, as);                                         // one predicated store, no branch
                gp += as ? 64u : 0u;
                kept |= bit;                                                   // the leaf's own particles always get a slot
                bit <<= 1;
                ++Cu;
                ++Cs;
            }
        }
    }
    C = (int)Cu;
    if (lane < fill && ((kept >> lane) & 1u)) S.cand[C0 + __popc(kept & ((1u << lane) - 1u))] = S.tidx[lane];
    g = (int)((gp - smem_u32(&S.queue[0][lane])) >> 6);
    return C;
}

__global__ void __launch_bounds__(LW * 32) k_nbr_lists(ListArgs a) {
    __shared__ WarpSmem sm[LW];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t leaf = (int64_t)blockIdx.x * LW + w;
    if (leaf >= a.nl) return;
    WarpSmem& S = sm[w];
    const int64_t i = leaf * CRK_LEAF + lane;
    const float4 pi = a.posh[i];
    const float xi = pi.x, yi = pi.y, zi = pi.z;
    const float hi2 = __fmul_rn(pi.w, pi.w);
    const float4 blo = a.leaf_lo[leaf], bhi = a.leaf_hi[leaf];
    const float hq2 = __fmul_rn(blo.w, blo.w);
    const uint32_t lt = (1u << lane) - 1u;
    int C = 0, g = 0, fill = 0;   // candidates of the segment, entries of this lane, staged candidates
    bool cwrap = false, wflag = false;   // wflag: this lane owns an entry of the segment that crosses the periodic boundary
    uint32_t prev = 0, first = 0;   // arena units of the previous / first segment header of this leaf

    auto put = [&](int slot, float x, float y, float z, float h2, uint32_t idx) {
        CRK_CHECK(a.flag, slot >= 0 && slot < CRK_TCULL + 2, 2);                           // cull tile slot
        float* fa = (float*)&S.ta[slot >> 1] + (slot & 1);
        float* fb = (float*)&S.tb[slot >> 1] + (slot & 1);
        fa[0] = -x; fa[2] = -y; fb[0] = -z; fb[2] = h2;
        S.tidx[slot] = idx;
    };
    auto emit = [&]() {
        const int K = __reduce_max_sync(0xffffffffu, g);
        const bool segwrap = __any_sync(0xffffffffu, wflag);
        const bool head = (prev == 0);   // a leaf's first segment keeps its candidates in the dense per-leaf array
        const unsigned long long cunits = head ? 0ull : (unsigned long long)((C + 3) >> 2);
        const unsigned long long units = CRK_SEG_HDR_UNITS + cunits + 4ull * K;
        unsigned long long base = 0;
        if (lane == 0) base = atomicAdd(a.counter, units);
        base = __shfl_sync(0xffffffffu, base, 0);
        // padding of shorter lanes: slot 0 (the sweeps prefetch it, never evaluate it) with the flag a gather sweep skips
        for (int k = g; k < K; ++k) S.queue[k][lane] = (uint16_t)CRK_ELL_SYM;
        __syncwarp();
        if (base + units <= a.arena_cap) {
            CRK_CHECK(a.flag, K <= CRK_QCAP && C <= CRK_CCAP && base >= 1, 3);                 // segment sizes
            uint4* hdr = a.arena + base;
            const uint32_t h1 = (uint32_t)C | (segwrap ? CRK_SEG_WRAP : 0u) | ((uint32_t)K << 16);
            if (lane == 0) hdr[0] = make_uint4(0u, h1, 0u, 0u);
            ((uint16_t*)(hdr + 1))[lane] = (uint16_t)g;
            uint32_t* cd = head ? a.cand_first + leaf * CRK_CAND_STRIDE : (uint32_t*)(hdr + CRK_SEG_HDR_UNITS);
            for (int c = lane; c < C; c += 32) cd[c] = S.cand[c];
            // the entry block is the queue as it stands: K rows of 32 u16 = 4 K units
            uint4* el = hdr + CRK_SEG_HDR_UNITS + cunits;
            const uint4* qs = (const uint4*)&S.queue[0][0];
            for (int q = lane; q < 4 * K; q += 32) el[q] = qs[q];
            if (head) {
                if (lane == 0) a.seg_first[leaf] = make_uint4(0u, h1, 0u, (uint32_t)base);
                a.leaf_cnt[leaf * 32 + lane] = (uint16_t)g;
                first = (uint32_t)base;
            } else if (lane == 0) {
                ((uint32_t*)(a.arena + prev))[0] = (uint32_t)base;
                if (prev == first) ((uint32_t*)(a.seg_first + leaf))[0] = (uint32_t)base;
            }
            prev = (uint32_t)base;
        }   // else: arena overflow -- the host re-runs the kernel with a larger arena; the counter keeps the total need
        C = 0; g = 0; wflag = false;
        __syncwarp();
    };
    // a leaf that straddles the periodic boundary needs the wrap in its own tile too
    const bool selfwrap = (bhi.x - blo.x > a.half) || (bhi.y - blo.y > a.half) || (bhi.z - blo.z > a.half);
    auto flush = [&](bool selftile) {
        const int maxlen = __reduce_max_sync(0xffffffffu, g);
        if (C + fill > CRK_CCAP || maxlen + fill > CRK_QCAP) emit();
        if ((fill & 1) && lane == 0) put(fill, 3.0e30f, 3.0e30f, 3.0e30f, 0.0f, 0u);
        __syncwarp();
        if (selftile && selfwrap) C = test_tile<true, true>(S, a.flag, fill, C, g, wflag, lane, xi, yi, zi, hi2, a.L, a.half);
        else if (selftile) C = test_tile<false, true>(S, a.flag, fill, C, g, wflag, lane, xi, yi, zi, hi2, a.L, a.half);
        else if (cwrap) C = test_tile<true, false>(S, a.flag, fill, C, g, wflag, lane, xi, yi, zi, hi2, a.L, a.half);
        else C = test_tile<false, false>(S, a.flag, fill, C, g, wflag, lane, xi, yi, zi, hi2, a.L, a.half);
        fill = 0;
        cwrap = false;
        __syncwarp();
    };

    const uint64_t e0 = (uint64_t)leaf * a.cap, e1 = e0 + min(a.cnt[leaf], a.cap);   // an overflowed list is rebuilt by the host
    uint32_t ent = (e0 < e1) ? a.list[e0] : 0u;
    float4 pj = (e0 < e1) ? a.posh[(int64_t)(ent & CRK_LEAF_MASK) * CRK_LEAF + lane] : make_float4(0, 0, 0, 0);
    // the query leaf itself goes first and keeps all 32 particles: slots 0..31 of the first segment are the leaf's own
    // particles in lane order, so a sweep finds the i-state of its lanes in the tile it stages anyway
    put(lane, xi, yi, zi, hi2, (uint32_t)i);
    fill = 32;
    flush(true);
    for (uint64_t e = e0; e < e1; ++e) {
        const uint32_t cur = ent;
        const float4 pc = pj;
        if (e + 1 < e1) {   // prefetch the next leaf's positions
            ent = a.list[e + 1];
            pj = a.posh[(int64_t)(ent & CRK_LEAF_MASK) * CRK_LEAF + lane];
        }
        const int64_t b = (int64_t)(cur & CRK_LEAF_MASK);
        CRK_CHECK(a.flag, b < a.nl, 4);                                                        // leaf-list entry
        const bool wrap = (cur & CRK_FLAG_WRAP) != 0;
        float gx, gy, gz;
        if (!wrap) {
            gx = gap1(blo.x, bhi.x, pc.x); gy = gap1(blo.y, bhi.y, pc.y); gz = gap1(blo.z, bhi.z, pc.z);
        } else {
            gx = gap1_wrap(blo.x, bhi.x, pc.x, a.L); gy = gap1_wrap(blo.y, bhi.y, pc.y, a.L); gz = gap1_wrap(blo.z, bhi.z, pc.z, a.L);
        }
        const float g2 = __fmaf_rn(gz, gz, __fmaf_rn(gy, gy, __fmul_rn(gx, gx)));
        const float hj2 = __fmul_rn(pc.w, pc.w);
        const bool surv = g2 < fmaxf(hq2, hj2);
        const uint32_t m = __ballot_sync(0xffffffffu, surv);
        const int cnt = __popc(m);
        if (cnt == 0) continue;
        if (b == leaf) continue;                                         // done first
        if (fill + cnt > CRK_TCULL) flush(false);
        if (surv) put(fill + __popc(m & lt), pc.x, pc.y, pc.z, hj2, (uint32_t)(b * CRK_LEAF + lane));
        cwrap = cwrap || wrap;
        fill += cnt;
    }
    if (fill > 0) flush(false);
    if (C > 0) emit();
    if (prev == 0 && lane == 0) a.seg_first[leaf] = make_uint4(0u, 0u, 0u, 0u);
}

__global__ void k_set_u64(unsigned long long* p, unsigned long long v) { *p = v; }

}  // namespace

// launches the builder; the arena need (status word FW_ARENA) is checked by crk_build_cells at its single synchronisation
int crk_build_nbr_lists(crk_ctx* c) {
    const int64_t nl = c->nl;
    CRK_TRY(crk_ensure(c, c->seg_first, (size_t)(nl + 1) * sizeof(uint4)));
    CRK_TRY(crk_ensure(c, c->leaf_cnt, (size_t)(nl + 1) * 32 * sizeof(uint16_t)));
    CRK_TRY(crk_ensure(c, c->cand_first, (size_t)(nl + 1) * CRK_CAND_STRIDE * sizeof(uint32_t)));
    // first guess: ~6 KB per leaf at ~60 neighbours; grown to the exact need if the builder reports more
    if (!c->arena.p) CRK_TRY(crk_ensure(c, c->arena, (size_t)nl * 6656 + 65536));
    unsigned long long* d_counter = (unsigned long long*)((int*)c->flag.p + FW_ARENA);
    ListArgs a;
    a.n = c->n; a.nl = nl; a.L = c->prm.box; a.half = 0.5f * c->prm.box;
    a.cnt = (const uint32_t*)c->nbr_cnt.p; a.list = (const uint32_t*)c->nbr_list.p; a.cap = (uint32_t)c->leaf_list_cap;
    a.posh = (const float4*)c->posh.p; a.leaf_lo = (const float4*)c->leaf_lo.p; a.leaf_hi = (const float4*)c->leaf_hi.p;
    a.arena = (uint4*)c->arena.p;
    a.arena_cap = crk_arena_cap_units(c);
    a.counter = d_counter;
    a.seg_first = (uint4*)c->seg_first.p;
    a.leaf_cnt = (uint16_t*)c->leaf_cnt.p;
    a.cand_first = (uint32_t*)c->cand_first.p;
    a.flag = (int*)c->flag.p;
    k_set_u64<<<1, 1, 0, c->stream>>>(d_counter, 1ull);
    CRK_TRY(crk_check_launch(c, "k_set_u64"));
    k_nbr_lists<<<(unsigned)((nl + LW - 1) / LW), LW * 32, 0, c->stream>>>(a);
    return crk_check_launch(c, "k_nbr_lists");
}

// usable arena units: the sweeps prefetch entry rows a little beyond a segment, so a tail margin stays free; segment links
// are 32-bit unit indices (64 GB)
unsigned long long crk_arena_cap_units(const crk_ctx* c) {
    unsigned long long cap = (unsigned long long)(c->arena.cap / 16);
    cap = cap > 256 ? cap - 256 : 0;
    return cap > 0xffffffffull ? 0xffffffffull : cap;
}
