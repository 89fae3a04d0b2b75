// lbm_stage.cuh -- the warp-specialised, shared-memory-staged stream-collide kernel for sm_100a: the same time step
// as stream_collide_kernel (Listing 2; eqs (24)-(28)), with BOTH the DDF
// loads and the DDF stores moved by the bulk-copy engine (cp.async.bulk, SASS UBLKCP), so that the arithmetic warps
// execute no global-memory instruction and no 64-bit address arithmetic on the way.
//
// Why (profiles/r01e_round1_final.md, profiles/r02a_staged_kernel.md): the first staged kernel (lbm_bulk.cuh) spent,
// of 374 lane-instructions per cell (FP16S), 19 on 64-bit store addresses and ~50 on tile bookkeeping and copy issue
// that every warp repeated; a cell pair with a flag bit dragged its whole warp through the slow path.  Here
//   * one LOADER warp per CTA issues the bulk loads of a tile -- one contiguous segment per direction, because a tile
//     is a run of consecutive cells and the layout is structure-of-arrays -- into an input stage,
//     and one STORER warp sends a computed tile from an output stage to B the same way;
//   * 14 consumer warps only read shared memory, collide and write shared memory; every address is "thread base +
//     immediate".  A tile is cut into chunks of 32 cell pairs; a warp that is free takes the CTA's next chunk (one
//     shared-memory counter), so the warps stay evenly loaded whatever the tile size and whatever else a warp has to do
//     (the list pass below).  Stages are handed over by mbarriers (full / in_empty / out_full / out_empty), on which
//     every chunk arrives once; there is no CTA-wide barrier in the loop;
//   * the main pass knows NO flags: every cell of a tile is pulled, collided and stored as if it were fluid.  The
//     flagged cells -- walls and equilibrium boundaries, which the step must leave untouched (R15), and
//     the cells next to a wall (halfway bounce-back R3, moving wall R9) -- are put right afterwards: lbm_set_flags
//     compacts them into per-tile lists, and a few tiles later, once the tile's bulk store is complete, the warps that
//     take the chunks of a tile also walk an equal share of an earlier tile's list, one cell per lane: a fixed cell gets
//     its values copied back from A, a cell next to a wall is recomputed from A with its bounce-back links and stored
//     again.  The list pass works on global memory only, so it holds no stage, and a warp busy with it simply takes
//     fewer chunks; a tile without flagged cells costs one compare.
// Arithmetic, operation order and codecs are those of lbm_lattice.cuh / lbm_codecs.cuh: the stored results are
// bit-identical to stream_collide_kernel's and to the oracle's.
#pragma once
#include "lbm_bulk.cuh"

namespace lbmk {

// shared -> global, completion tracked by the issuing thread's bulk async-group
__device__ __forceinline__ void bulk_s2g(void *dst, unsigned src, unsigned bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() {       // all but the N newest groups have finished READING shared memory
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
template <int N>
__device__ __forceinline__ void bulk_wait() {            // all but the N newest groups are complete (written)
    asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory");
}
// Orders this thread's accesses through the async proxy (the bulk-copy engine) and through the generic proxy (ordinary
// loads / stores) to the same GLOBAL addresses.  The list pass overwrites, with ordinary stores, cells that a bulk store
// wrote: without the fence on the way from "the bulk store is complete" to "the ordinary store is issued" the bulk
// store's data can still land last (seen on FP32 boxes, whose stores drain slowest: about one tile in 2*10^7).
__device__ __forceinline__ void fence_async_global() { asm volatile("fence.proxy.async.global;" ::: "memory"); }

// ---- compile-time shape ----------------------------------------------------------------------------
// One CTA of 16 warps per SM -- four per scheduler, 128 registers per thread, which the two-cell collision needs --
// one loader, one storer, 14 consumers.  A tile is up to TC cells = TC/64 chunks of 32 cell pairs, one pair per lane.
template <int Q, int F, int ALT = 0>
struct StageShape {
    typedef Elem<F> E;
    static constexpr int ES = E::SIZE;                      // bytes per stored DDF
    static constexpr int PAD = 16;                          // halo pad in front of and behind every input segment
    static constexpr int LIMIT = 227 * 1024 - 1024;         // one CTA per SM
    static constexpr int TABB = PairCodec<F>::TABLE ? 512 * 16 : 0;
    // rings: tile headers (16 bytes each), "tile stored" barriers.  A `done` barrier is waited on by phase parity, so a
    // waiter must test it before its slot has completed a second time, i.e. before the storer is DONES + WLAG - LAG tiles
    // past the waiter's tile: 15 tiles with 16 slots, far beyond what the stage hand-over lets the warps drift apart
    static constexpr int HDRS = 16, DONES = 16;
    static constexpr int in_bytes(int tc) { return Q * (tc * ES + 2 * PAD); }
    static constexpr int out_bytes(int tc) { return Q * tc * ES; }
    static constexpr int need(int tc, int si, int so) { return si * in_bytes(tc) + so * out_bytes(tc) + TABB + HDRS * 16 + 256; }
    // cells per tile: the largest of 2048 / 1024 / 768 that leaves room for THREE input stages (16-bit D2Q9: 2048, D3Q19:
    // 1024, D3Q27: 768), else the largest that fits with two (FP32).  Measured: the third input stage
    // is worth more than a larger tile -- unless the box's rows fill the smaller tile badly.  HAS_ALT: where the two-stage
    // shape holds more cells (D3Q27 16-bit: 1024), it is compiled as well (ALT = 1) and stage_alt() (lbm_unit.cu) picks
    // per box.
    static constexpr int TC3 = need(2048, 3, 2) <= LIMIT ? 2048 : need(1024, 3, 2) <= LIMIT ? 1024 : need(768, 3, 2) <= LIMIT ? 768 : 0;
    static constexpr int TC2 = need(1024, 2, 2) <= LIMIT ? 1024 : need(512, 2, 2) <= LIMIT ? 512 : 256;
    static constexpr bool HAS_ALT = TC3 != 0 && TC2 > TC3;
    static constexpr int TC = (TC3 != 0 && !(ALT == 1 && HAS_ALT)) ? TC3 : TC2;
    static constexpr int S_OUT = 2;                                                     // output stages
    static constexpr int S_IN = need(TC, 3, S_OUT) <= LIMIT ? 3 : 2;                    // input stages
    // consumer warps: 14 (+ loader + storer = 16 warps, 128 registers per thread).  The D3Q19 posits run 18 + 2 warps of 96
    // registers instead: their encoder-table reads keep the shared-memory pipe 79% busy and the warps waiting on it
    // (profiles/r02b_staged_kernels.md), and four more warps hide more of that than the 40 spilled bytes cost (+4-8%)
    static constexpr bool MANY = PairCodec<F>::TABLE && !PairCodec<F>::FAST && Q == 19;
    static constexpr int NCW = MANY ? 18 : 14;
    // D3Q27's two cells of 27 populations do not fit 128 registers together (124 bytes of spills): there -- and in the
    // 96-register posit kernels -- a thread finishes its first cell (pull, collide, encode, half-word stores) before it
    // pulls the second
    static constexpr bool SPLIT = Q == 27 || MANY;
    // chunk ids a warp takes at a time.  The per-claim work (the counter, two barrier waits, the header, two arrivals, the
    // list-pass test) is about 40 of the 120 non-arithmetic warp-instructions per chunk: against D2Q9's nine directions that
    // is a tenth of the kernel, and its 2048-cell tiles have 32 chunks, so two at a time still leave 16 claims per tile.
    // D3Q19 (16 chunks per tile, 14 warps) loses 5-10% on 256^3 boxes with two: one there.
    static constexpr int CPC = (Q == 9 && ES == 2) ? 2 : 1;
    static constexpr int NCT = 32 * NCW, NT = NCT + 64;                                 // + the loader and the storer warp
    // The storer reports tile k written WLAG tiles later, and the list pass of a tile runs LAG = WLAG + 1 tiles after it,
    // together with the lists of its group of LG consecutive tiles.  Both are as SHORT as they can be: the list pass
    // re-reads, sector by sector, values that the main pass streamed through L2 a moment ago, and the sooner it comes the
    // more of them are still there -- cavity 256^3, WLAG = 3 -> 0: FP32 32.1 -> 35.5, FP16S 50.9 -> 54.9 GLUPs/s, although the
    // storer now waits for each tile's writes before it sends the next.  Grouping fills the lanes of the warps that
    // walk the lists (a cavity tile has a dozen listed cells): LG = 4 gives the instruction-bound formats +24% (FP16C) to
    // +34% (P16_1S); the lighter kernels (FP32, FP16S, FP16), which feel the re-reads more, are best with 2 (FP16S 58.0
    // against 54.8 with 4 and 52.7 with 1; FP32 37.4 against 35.5 with 1).
    static constexpr int WLAG = 0;
    static constexpr int LAG = WLAG + 1;
    static constexpr int LG = (ES == 4 || F == F_FP16S || F == F_FP16) ? 2 : 4;
    static constexpr int ROWB = TC * ES + 2 * PAD;          // one direction of one input stage
    static constexpr int INB = in_bytes(TC);
    static constexpr int OPITCH = TC * ES;                  // one direction of one output stage
    static constexpr int OUTB = out_bytes(TC);
    static constexpr int OUT_OFF = S_IN * INB;
    static constexpr int TAB_OFF = OUT_OFF + S_OUT * OUTB;
    static constexpr int HDR_OFF = TAB_OFF + TABB;
    static constexpr int BAR_OFF = HDR_OFF + HDRS * 16;     // full[S_IN], in_empty[S_IN], out_full[S_OUT], out_empty[S_OUT], done[DONES]
    static constexpr int CTR_OFF = BAR_OFF + (2 * (S_IN + S_OUT) + DONES) * 8;          // the chunk counter
    static constexpr int SMEM = CTR_OFF + 8;
    static_assert(NT == (MANY ? 640 : 512), "16 warps: 128 registers per thread (20: 96)");
    static_assert(SMEM <= LIMIT, "the CTA must fit one SM");
    static_assert(INB % 16 == 0 && ROWB % 16 == 0 && OUTB % 16 == 0 && TAB_OFF % 16 == 0 && BAR_OFF % 8 == 0, "alignment");
    static_assert((2 * (S_IN + S_OUT) + DONES) * 8 + 8 <= 256, "the barriers fit the 256 bytes need() reserves for them");
    static_assert(LAG + LG - 1 + S_IN + 2 < HDRS && LAG + LG <= DONES, "ring sizes");
    static_assert(S_OUT >= 2, "the chunk-wise hand-over of the output stages needs two of them");
};

// The value of direction I for ONE of the thread's two cells (J = 0: cell xl, J = 1: cell xl+1) from the staged segment.
//   own = address of element xl of direction 0's segment; left = element "xl - 1", right = element "xl + 2" (already
//   wrapped / pointing into the pads); direction I adds the immediate I * ROWB.
// A direction without an x component is one aligned load for both cells: cell 0's pull keeps the raw word in w[I] for
// cell 1's.
template <int Q, int F, int ALT, class PC, int J, int I>
struct PullCell {
    typedef StageShape<Q, F, ALT> SH;
    // accw / accs collect the raw words / single codes for PairCodec<F>::CHECK
    static __device__ __forceinline__ void run(const char *own, const char *left, const char *right, float (&f)[Q], unsigned (&w)[Q],
                                               unsigned &accw, unsigned &accs) {
        typedef Lat<Q> L;
        constexpr int cx = L::c(I, 0);
        constexpr int o = I * SH::ROWB;
        if constexpr (SH::ES == 4) {
            if (cx == 0) {
                if (J == 0) {
                    const float2 v = *reinterpret_cast<const float2 *>(own + o);
                    f[I] = v.x;
                    w[I] = __float_as_uint(v.y);
                } else {
                    f[I] = __uint_as_float(w[I]);
                }
            } else if (cx > 0) {              // sources xl-1, xl
                f[I] = lds_f32(J == 0 ? left + o : own + o);
            } else {                          // sources xl+1, xl+2
                f[I] = lds_f32(J == 0 ? own + o + 4 : right + o);
            }
        } else {
            if (cx == 0) {
                if (J == 0) w[I] = lds_u32(own + o);
                if (PC::CHECK) accw |= w[I];
                float a, b;
                PC::dec2(w[I], a, b);
                f[I] = J == 0 ? a : b;
            } else {
                const char *at = cx > 0 ? (J == 0 ? left + o : own + o) : (J == 0 ? own + o + 2 : right + o);
                const int c = PC::SEXT ? lds_s16(at) : lds_u16(at);      // (sign-extended only where the decoder wants it)
                if (PC::CHECK) accs |= (unsigned)c;
                f[I] = PC::dec1(c);
            }
        }
        PullCell<Q, F, ALT, PC, J, I + 1>::run(own, left, right, f, w, accw, accs);
    }
};
template <int Q, int F, int ALT, class PC, int J>
struct PullCell<Q, F, ALT, PC, J, Q> {
    static __device__ __forceinline__ void run(const char *, const char *, const char *, float (&)[Q], unsigned (&)[Q], unsigned &,
                                               unsigned &) {}
};

// One cell's pull with the format's cheap decoders, again with the full-range ones if a code outside their domain
// shows up (posits: PairCodec<F>::CHECK; `wide` = the warp is in full-range mode already).  Returns whether such a
// code was met.
template <int Q, int F, int ALT, int J>
__device__ __forceinline__ bool pull_cell(const char *own, const char *left, const char *right, float (&f)[Q], unsigned (&w)[Q], bool wide) {
    typedef PairCodec<F> PC;
    unsigned accw = 0, accs = 0;
    if constexpr (PC::CHECK != 0) {
        if (!wide) PullCell<Q, F, ALT, PC, J, 0>::run(own, left, right, f, w, accw, accs);
        if (wide || (((accw >> (16 * J)) | accs) & PC::CHECK) != 0) {
            accw = accs = 0;
            PullCell<Q, F, ALT, FullRange<F>, J, 0>::run(own, left, right, f, w, accw, accs);
        }
        return (((accw >> (16 * J)) | accs) & PC::CHECK) != 0;
    } else {
        PullCell<Q, F, ALT, PC, J, 0>::run(own, left, right, f, w, accw, accs);
        return false;
    }
}

// ---- loader: tile t into an input stage -------------------------------------------------------------------
// The segment of source row (y - c_iy, z - c_iz) of every direction i (periodic wrap in y and z is a different row
// address, R2).  Everything here is warp-uniform (the bulk-copy instruction takes uniform operands); lane 0 issues.
// Away from the box faces a direction's source is "tile base + per-direction constant" (BulkGeom::src_boff, in the
// kernel's constant bank): one copy per direction for a tile of whole rows, one copy plus a 16-byte halo copy (the
// element before / after the segment, for the directions shifted in x) for a segment of a long row.
template <int Q, int F, int ALT, int I>
struct LoadDir {
    typedef StageShape<Q, F, ALT> SH;
    static __device__ __forceinline__ void run(const char *A, const Params &p, const BulkGeom &g, const TileCoord &c, bool single,
                                               bool face, long long first_b, unsigned stage, unsigned full) {
        typedef Lat<Q> L;
        constexpr int ES = SH::ES, cx = L::c(I, 0), cy = L::c(I, 1), cz = L::c(I, 2);
        const unsigned dst = stage + I * SH::ROWB + SH::PAD;
        const unsigned rowb = (unsigned)(c.w * ES);
        if (!face || (cy == 0 && cz == 0)) {
            // no wrap: the tile's own address plus the direction's constant
            const char *src = A + first_b + g.src_boff[I];
            bulk_g2s(dst, src, (unsigned)c.rows * rowb, full);
            if (!single && cx > 0) bulk_g2s(dst - SH::PAD, src + (c.x0 == 0 ? (long long)p.nx * ES : 0) - SH::PAD, SH::PAD, full);
            if (!single && cx < 0) bulk_g2s(dst + rowb, src + rowb - (c.x0 + c.w == p.nx ? (long long)p.nx * ES : 0), SH::PAD, full);
        } else {
            int zs = c.z - cz;
            zs = zs < 0 ? p.nz - 1 : zs >= p.nz ? 0 : zs;
            const char *plane = A + g.dir_boff[I] + (long long)p.nx * p.ny * zs * ES + (long long)c.x0 * ES;
            const long long pitch = (long long)p.nx * ES;
            const int ys = c.y - cy;                                         // source row of the tile's first row
            // per direction the source rows are one run, or two where the tile's first / last row wraps in y
            if (ys < 0) {                                                    // first row from the opposite face
                bulk_g2s(dst, plane + pitch * (p.ny - 1), rowb, full);
                if (c.rows > 1) bulk_g2s(dst + rowb, plane, (c.rows - 1) * rowb, full);
            } else if (ys + c.rows > p.ny) {                                 // last row from the opposite face
                if (c.rows > 1) bulk_g2s(dst, plane + pitch * ys, (c.rows - 1) * rowb, full);
                bulk_g2s(dst + (c.rows - 1) * rowb, plane, rowb, full);
            } else {
                bulk_g2s(dst, plane + pitch * ys, c.rows * rowb, full);
            }
            if (!single && cx != 0) {                                        // (a segment is one row)
                const int yw = ys < 0 ? p.ny - 1 : ys >= p.ny ? 0 : ys;
                const char *row = plane + pitch * yw - (long long)c.x0 * ES; // start of the source row
                if (cx > 0) bulk_g2s(dst - SH::PAD, row + (long long)(c.x0 == 0 ? p.nx : c.x0) * ES - SH::PAD, SH::PAD, full);
                else bulk_g2s(dst + rowb, row + (long long)(c.x0 + c.w == p.nx ? 0 : c.x0 + c.w) * ES, SH::PAD, full);
            }
        }
        LoadDir<Q, F, ALT, I + 1>::run(A, p, g, c, single, face, first_b, stage, full);
    }
};
template <int Q, int F, int ALT>
struct LoadDir<Q, F, ALT, Q> {
    static __device__ __forceinline__ void run(const char *, const Params &, const BulkGeom &, const TileCoord &, bool, bool, long long, unsigned,
                                               unsigned) {}
};

// hdr = the tile's slot in the header ring
template <int Q, int F, int ALT>
__device__ __forceinline__ void stage_issue_loads(const typename Elem<F>::T *__restrict__ A, const Params &p, const BulkGeom &g,
                                                  int t, unsigned lo, unsigned hi, unsigned stage, unsigned full, unsigned hdr, bool leader) {
    typedef StageShape<Q, F, ALT> SH;
    constexpr int ES = SH::ES;
    constexpr int n_shift = (Q == 9 ? 6 : Q == 19 ? 10 : 18);               // directions with c_x != 0
    const bool single = g.tiles_per_row == 1;
    const TileCoord c = tile_coord(t, g, p);
    const int cells = c.rows * c.w;
    if (!leader) return;
    // the tile's header for the consumer warps: cell pairs, and the tile's slice [lo, hi) of the flagged-cell list (the
    // caller read it a tile ahead: a load here would delay every tile's copies by a trip to memory).  Written before the
    // arrival below (release), read after the consumers' wait on the same barrier (acquire)
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(hdr), "r"((unsigned)(cells >> 1)), "r"(lo), "r"(hi), "r"(0u) : "memory");
    mbar_arrive_expect_tx(full, (unsigned)(Q * cells * ES + (single ? 0 : n_shift * SH::PAD)));
    const long long first_b = ((long long)p.nx * (c.y + (long long)p.ny * c.z) + c.x0) * ES;
    // tiles on a y or z face of the box pull some directions from the opposite face (R2)
    const bool face = c.y == 0 || c.y + c.rows == p.ny || c.z == 0 || c.z == p.nz - 1;
    LoadDir<Q, F, ALT, 0>::run(reinterpret_cast<const char *>(A), p, g, c, single, face, first_b, stage, full);
}

// ---- the list pass: one flagged cell, from and to global memory ------------------------------------------------
// The pull of direction I for a cell next to a wall: the links in `mask` bounce (R3), the others come
// from the neighbour.  The source ADDRESS is selected, not the load: all q loads are in flight together (a branch per
// direction would expose q memory latencies one after the other).
template <int Q, int F, int I>
struct PullMasked {
    typedef Elem<F> E;
    typedef typename E::T T;
    // copy_from >= 0: no pull at all -- the cell takes slot I of cell `copy_from` (a fixed cell: itself; an outflow cell:
    // its upstream neighbour), so that every kind of listed cell shares ONE batch of loads
    static __device__ __forceinline__ void run(const T *__restrict__ A, const Params &p, const long long (&rows)[3][3], int x, int xm,
                                               int xp, unsigned mask, long long copy_from, T (&raw)[Q]) {
        typedef Lat<Q> L;
        constexpr int cx = L::c(I, 0), cy = L::c(I, 1), cz = L::c(I, 2);
        const long long own = rows[1][1] + x;
        if (I == 0) {
            raw[0] = __ldg(A + (copy_from >= 0 ? copy_from : own));
        } else {
            const long long src = rows[1 - cy][1 - cz] + (cx == 0 ? x : cx > 0 ? xm : xp);
            const T *from_neighbour = A + (long long)I * p.N + src, *from_self = A + (long long)L::opp(I) * p.N + own;
            const T *from_copy = A + (long long)I * p.N + copy_from;
            raw[I] = __ldg(copy_from >= 0 ? from_copy : ((mask >> I) & 1u) ? from_self : from_neighbour);
        }
        PullMasked<Q, F, I + 1>::run(A, p, rows, x, xm, xp, mask, copy_from, raw);
    }
};
template <int Q, int F>
struct PullMasked<Q, F, Q> {
    typedef typename Elem<F>::T T;
    static __device__ __forceinline__ void run(const T *__restrict__, const Params &, const long long (&)[3][3], int, int, int, unsigned,
                                               long long, T (&)[Q]) {}
};
// R9: the moving-wall term of the bounced links of a cell one of whose walls moves (bit 31 of its mask)
template <int Q, int I>
struct MovingWallTerms {
    static __device__ __forceinline__ void run(const Params &p, const long long (&rows)[3][3], int x, int xm, int xp, unsigned mask,
                                               float (&f)[Q]) {
        typedef Lat<Q> L;
        constexpr int cx = L::c(I, 0), cy = L::c(I, 1), cz = L::c(I, 2);
        if ((mask >> I) & 1u) {
            const long long src = rows[1 - cy][1 - cz] + (cx == 0 ? x : cx > 0 ? xm : xp);
            const float uwx = __ldg(p.u0 + src), uwy = __ldg(p.u0 + p.N + src), uwz = __ldg(p.u0 + 2 * p.N + src);
            if (uwx != 0.0f || uwy != 0.0f || uwz != 0.0f)                   // rho_w = 1
                f[I] = add(f[I], mul(L::w6(I), cdot<Q, I>(uwx, uwy, uwz)));
        }
        MovingWallTerms<Q, I + 1>::run(p, rows, x, xm, xp, mask, f);
    }
};
template <int Q>
struct MovingWallTerms<Q, Q> {
    static __device__ __forceinline__ void run(const Params &, const long long (&)[3][3], int, int, int, unsigned, float (&)[Q]) {}
};

// fl = the cell's flag byte, mask = its `bounce` word.  A fixed cell (wall, equilibrium boundary: never updated,
// PAPER.md:1017; R15) gets the values it has in A back; an outflow cell (R18) the equilibrium of its upstream neighbour's
// moments; a cell next to a wall is computed again, this time with its bounce-back links, with the scalar converters
// (bit-identical to the pair converters: lbm_codec_pair_selftest).  The three kinds share their q loads and their q
// stores -- a warp whose lanes hold cells of several kinds (a row end: wall, neighbour of the wall) waits for memory once,
// only the arithmetic in between diverges.
template <int Q, int F, bool FORCE, int COLL>
__device__ __forceinline__ void fix_cell(const typename Elem<F>::T *__restrict__ A, typename Elem<F>::T *__restrict__ B, const Params &p,
                                         int x, int y, int z, unsigned fl, unsigned mask) {
    typedef Elem<F> E;
    typedef typename E::T T;
    const long long n = x + (long long)p.nx * (y + (long long)p.ny * z);
    const int ym = y == 0 ? p.ny - 1 : y - 1, yp = y == p.ny - 1 ? 0 : y + 1;
    const int zm = z == 0 ? p.nz - 1 : z - 1, zp = z == p.nz - 1 ? 0 : z + 1;
    const int ys[3] = {ym, y, yp}, zs[3] = {zm, z, zp};
    long long rows[3][3];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) rows[a][b] = (long long)p.nx * (ys[a] + (long long)p.ny * zs[b]);
    const int xm = x == 0 ? p.nx - 1 : x - 1, xp = x == p.nx - 1 ? 0 : x + 1;
    const long long copy_from = (fl & FLAG_FIXED) ? n : (fl & FLAG_OUT) ? n - x + xm : -1;
    T raw[Q];
    PullMasked<Q, F, 0>::run(A, p, rows, x, xm, xp, mask, copy_from, raw);
    if (!(fl & FLAG_FIXED)) {
        float f[Q];
#pragma unroll
        for (int i = 0; i < Q; ++i) {
            if constexpr (E::SIZE == 4) f[i] = raw[i];
            else f[i] = Codec<F>::dec((unsigned)raw[i]);
        }
        if (fl & FLAG_OUT) {                                                 // R18, as outflow_cell (lbm_kernels.cuh)
            float rho, j[3], u[3], feq[Q];
            moments<Q, true>(f, rho, j);
            const float Fv[3] = {p.fx, p.fy, p.fz};
#pragma unroll
            for (int a = 0; a < 3; ++a) u[a] = __fdiv_rn(FORCE ? fma_(-0.5f, Fv[a], j[a]) : j[a], rho);
            equilibrium<Q, true>(rho, u[0], u[1], u[2], feq);
#pragma unroll
            for (int i = 0; i < Q; ++i) f[i] = feq[i];
        } else {
            if (mask >> 31) MovingWallTerms<Q, 1>::run(p, rows, x, xm, xp, mask, f);
            collide<COLL, Q, FORCE>(f, p);
        }
#pragma unroll
        for (int i = 0; i < Q; ++i) {
            if constexpr (E::SIZE == 4) raw[i] = f[i];
            else raw[i] = (T)Codec<F>::enc(f[i]);
        }
    }
#pragma unroll
    for (int i = 0; i < Q; ++i) B[(long long)i * p.N + n] = raw[i];
}

// one flagged cell: entry e of the list of tile t
template <int Q, int F, bool FORCE, int COLL>
__device__ __forceinline__ void fix_list_entry(const typename Elem<F>::T *__restrict__ A, typename Elem<F>::T *__restrict__ B,
                                               const Params &p, const BulkGeom &g, int t, uint2 e) {
    const TileCoord c = tile_coord(t, g, p);
    const FastDiv by_hw = c.last ? g.by_hw_last : g.by_hw_full;
    const int ci = (int)(e.x & 0xFFFFu);                                     // cell index inside the tile
    const int r = by_hw.div(ci >> 1), xl = ci - r * c.w;
    fix_cell<Q, F, FORCE, COLL>(A, B, p, c.x0 + xl, c.y + r, c.z, e.x >> 16, e.y);
}

template <int Q, int F, bool FORCE, int COLL = 0, int ALT = 0>
__global__ void __launch_bounds__(StageShape<Q, F, ALT>::NT, 1)
stream_collide_staged_kernel(const typename Elem<F>::T *__restrict__ A, typename Elem<F>::T *__restrict__ B,
                             const __grid_constant__ Params p, const __grid_constant__ BulkGeom g,
                             const EncEntry *__restrict__ enc_table) {
    typedef StageShape<Q, F, ALT> SH;
    typedef Elem<F> E;
    typedef typename E::T T;
    constexpr int ES = SH::ES, S_IN = SH::S_IN, S_OUT = SH::S_OUT, NCW = SH::NCW, LAG = SH::LAG;
    typedef PairCodec<F> PC;
    constexpr int SC = PC::SC;

    extern __shared__ __align__(128) char smem[];
    const unsigned smem_base = smem_addr(smem);
    const unsigned bar_full = smem_base + SH::BAR_OFF, bar_in_empty = bar_full + S_IN * 8;
    const unsigned bar_out_full = bar_in_empty + S_IN * 8, bar_out_empty = bar_out_full + S_OUT * 8;
    const unsigned bar_done = bar_out_empty + S_OUT * 8;
    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);                  // warp-uniform by construction

    if (tid == 0) {
        for (int s = 0; s < S_IN; ++s) {
            mbar_init(bar_full + s * 8, 1);                                  // the loader's arrive.expect_tx
            mbar_init(bar_in_empty + s * 8, 1u << g.chunk_shift);            // one arrival per chunk id
        }
        for (int s = 0; s < S_OUT; ++s) {
            mbar_init(bar_out_full + s * 8, 1u << g.chunk_shift);
            mbar_init(bar_out_empty + s * 8, 1);                             // the storer, once its bulk stores have read the stage
        }
        for (int s = 0; s < SH::DONES; ++s) mbar_init(bar_done + s * 8, 1);  // the storer, once a tile is written
        *reinterpret_cast<unsigned *>(smem + SH::CTR_OFF) = 0u;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_async_smem();
    }
    const EncEntry *tab = reinterpret_cast<const EncEntry *>(smem + SH::TAB_OFF);
    if constexpr (PC::TABLE) {
        for (int i = tid; i < 512; i += SH::NT)
            reinterpret_cast<uint4 *>(smem + SH::TAB_OFF)[i] = __ldg(reinterpret_cast<const uint4 *>(enc_table) + i);
    }
    __syncthreads();

    const int stride = gridDim.x;
    const bool lists = p.fix_off != nullptr;

    if (warp == NCW) {
        // ================= the loader warp =================
        const bool leader = lane == 0;
        // the slice of the flagged-cell list of tile t, and the list entries on their way into L2 for the list pass
        auto list_slice = [&](long long t, unsigned &lo, unsigned &hi) {
            lo = hi = 0;
            if (lists && leader && t < g.n_tiles) {
                lo = __ldg(p.fix_off + t);
                hi = __ldg(p.fix_off + t + 1);
            }
        };
        auto list_prefetch = [&](unsigned lo, unsigned hi) {
            if (leader && lo < hi) {
                const char *a = reinterpret_cast<const char *>(p.fix_cells + lo), *b = reinterpret_cast<const char *>(p.fix_cells + hi);
#pragma unroll 1
                for (int n = 0; a < b && n < 8; a += 128, ++n) asm volatile("prefetch.global.L2 [%0];" ::"l"(a));
            }
        };
        int k = 0;
        unsigned lo, hi;
        list_slice(blockIdx.x, lo, hi);
#pragma unroll 1
        for (; k < S_IN; ++k) {                                              // prologue: fill every input stage
            const long long t = (long long)blockIdx.x + (long long)k * stride;
            if (t < g.n_tiles)
                stage_issue_loads<Q, F, ALT>(A, p, g, (int)t, lo, hi, smem_base + k * SH::INB, bar_full + k * 8, smem_base + SH::HDR_OFF + (k % SH::HDRS) * 16, leader);
            list_prefetch(lo, hi);
            list_slice(t + stride, lo, hi);
        }
        int si = 0;
        unsigned ph_in = 0;
#pragma unroll 1
        for (long long tn = (long long)blockIdx.x + (long long)S_IN * stride; tn < g.n_tiles; tn += stride, ++k) {
            // refill the input stage of tile k - S_IN with tile k once every consumer warp has its values out of it
            mbar_wait(bar_in_empty + si * 8, ph_in);
            stage_issue_loads<Q, F, ALT>(A, p, g, (int)tn, lo, hi, smem_base + si * SH::INB, bar_full + si * 8, smem_base + SH::HDR_OFF + (k % SH::HDRS) * 16, leader);
            list_prefetch(lo, hi);
            list_slice(tn + stride, lo, hi);                                 // the next tile's, in flight while this warp waits
            if (++si == S_IN) { si = 0; ph_in ^= 1u; }
        }
        return;
    }
    if (warp == NCW + 1) {
        // ================= the storer warp: a computed tile leaves as one contiguous segment per direction; the output
        // stage is handed back as soon as the bulk-copy engine has read it, the tile is reported written one tile later
        const bool leader = lane == 0;
        int so = 0, k = 0;
        unsigned ph_out = 0;
#pragma unroll 1
        for (int t = blockIdx.x; t < g.n_tiles; t += stride, ++k) {
            mbar_wait(bar_out_full + so * 8, ph_out);
            const TileCoord c = tile_coord(t, g, p);
            char *first = reinterpret_cast<char *>(B) + ((long long)p.nx * (c.y + (long long)p.ny * c.z) + c.x0) * ES;
            const unsigned bytes = (unsigned)(c.rows * c.w * ES);
            const unsigned ostage = smem_base + SH::OUT_OFF + so * SH::OUTB;
            if (leader) {
#pragma unroll
                for (int i = 0; i < Q; ++i) bulk_s2g(first + g.dir_boff[i], ostage + i * SH::OPITCH, bytes);
                bulk_commit();
                bulk_wait_read<0>();
                mbar_arrive(bar_out_empty + so * 8);
                if (lists && k >= SH::WLAG) {
                    bulk_wait<SH::WLAG>();                                   // tile k - WLAG is written
                    fence_async_global();
                    mbar_arrive(bar_done + ((k - SH::WLAG) % SH::DONES) * 8);
                }
            }
            __syncwarp();
            if (++so == S_OUT) { so = 0; ph_out ^= 1u; }
        }
        if (leader) {
            bulk_wait<0>();                                                  // all stores complete before the CTA's shared memory goes
            fence_async_global();
            if (lists)
                for (int j = k > SH::WLAG ? k - SH::WLAG : 0; j < k; ++j) mbar_arrive(bar_done + (j % SH::DONES) * 8);
        }
        return;
    }

    // ================= consumer warps =================
    const bool single = g.tiles_per_row == 1;            // a tile spans its rows: x wraps inside the segment
    bool full_mode = false;                              // posits: this thread currently needs the full-range decoders
    const int hw = g.tile_w >> 1;
    const int shift = g.chunk_shift;
    const int my_tiles = (g.n_tiles - (int)blockIdx.x + stride - 1) / stride;           // tiles of this CTA
    // chunk ids: tile k of this CTA has the ids [k << shift, (k + 1) << shift); LAG more "tiles" without cells carry the
    // list passes of the last LAG tiles
    const unsigned n_ids = (unsigned)(my_tiles + (lists ? LAG : 0)) << shift;
    unsigned *counter = reinterpret_cast<unsigned *>(smem + SH::CTR_OFF);
#pragma unroll 1
    for (;;) {
        unsigned id = 0;
        if (lane == 0) id = atomicAdd(counter, (unsigned)SH::CPC);           // ids id .. id + CPC - 1, all of one tile (2^shift >= 8)
        id = __shfl_sync(0xffffffffu, id, 0);
        if (id >= n_ids) break;
        const int k = (int)(id >> shift), c0 = (int)(id & ((1u << shift) - 1u));
        if (k < my_tiles) {
            const int si = k % S_IN, so = k % S_OUT;
            const char *stage = smem + si * SH::INB;
            char *ostage = smem + SH::OUT_OFF + so * SH::OUTB;
            mbar_wait(bar_full + si * 8, (unsigned)(k / S_IN) & 1u);
            const int pairs = *reinterpret_cast<const int *>(smem + SH::HDR_OFF + (k % SH::HDRS) * 16);   // the loader wrote it
            // the bulk stores of tile k - S_OUT have read this output stage.  (A chunk id without cells waits too: its
            // arrival below must not count for the stage's previous use.)  Waiting here, not between the collision and
            // the stores, lets every result go to shared memory as soon as it exists.
            if (k >= S_OUT) mbar_wait(bar_out_empty + so * 8, (unsigned)(k / S_OUT - 1) & 1u);
#pragma unroll 1
            for (int c = c0; c < c0 + SH::CPC; ++c) {
            const int fp = 32 * c + lane;
            if (32 * c < pairs) {
                // the pair's place in a direction's segment and in the row (only the row ends matter: x wraps)
                int xl = 2 * fp;
                if (single) xl = 2 * (fp - g.by_hw_full.div(fp) * hw);
                const int own_b = SH::PAD + 2 * fp * ES;
                const int left_b = own_b - ES + ((single && xl == 0) ? g.tile_w * ES : 0);             // element "xl - 1" (wrapped)
                const int right_b = own_b + 2 * ES - ((single && xl + 2 == g.tile_w) ? g.tile_w * ES : 0);   // element "xl + 2"
                bool warp_full = false;
                if constexpr (PC::CHECK != 0) warp_full = __any_sync(0xffffffffu, full_mode);   // one decoder per warp where possible
                if constexpr (SH::SPLIT) {
                    if (fp < pairs) {
                        float f[Q];
                        unsigned wd[Q];
                        char *o = ostage + 2 * fp * ES;
                        full_mode = pull_cell<Q, F, ALT, 0>(stage + own_b, stage + left_b, stage + right_b, f, wd, warp_full);
                        collide<COLL, Q, FORCE, SC, ES == 2 ? 1 : 2>(f, p);
                        if constexpr (PC::FAST) {                           // (the table-free encoder, as in the pair path below)
                            unsigned acc = full_mode ? PC::FAST_BAD : 0u;
                            if (!full_mode) {
#pragma unroll
                                for (int i = 0; i < Q; ++i) *reinterpret_cast<unsigned short *>(o + i * SH::OPITCH) = (unsigned short)PC::enc1_fast(f[i], acc);
                            }
                            if (acc & PC::FAST_BAD) {
#pragma unroll
                                for (int i = 0; i < Q; ++i) *reinterpret_cast<unsigned short *>(o + i * SH::OPITCH) = (unsigned short)PC::enc1(f[i], tab);
                            }
                        } else {
#pragma unroll
                            for (int i = 0; i < Q; ++i) {
                                if constexpr (ES == 4) *reinterpret_cast<float *>(o + i * SH::OPITCH) = f[i];
                                else *reinterpret_cast<unsigned short *>(o + i * SH::OPITCH) = (unsigned short)PC::enc1(f[i], tab);
                            }
                        }
                        full_mode |= pull_cell<Q, F, ALT, 1>(stage + own_b, stage + left_b, stage + right_b, f, wd, warp_full);
                        collide<COLL, Q, FORCE, SC, ES == 2 ? 1 : 2>(f, p);
                        if constexpr (PC::FAST) {                           // (the table-free encoder, as in the pair path below)
                            unsigned acc = full_mode ? PC::FAST_BAD : 0u;
                            if (!full_mode) {
#pragma unroll
                                for (int i = 0; i < Q; ++i) *reinterpret_cast<unsigned short *>(o + i * SH::OPITCH + 2) = (unsigned short)PC::enc1_fast(f[i], acc);
                            }
                            if (acc & PC::FAST_BAD) {
#pragma unroll
                                for (int i = 0; i < Q; ++i) *reinterpret_cast<unsigned short *>(o + i * SH::OPITCH + 2) = (unsigned short)PC::enc1(f[i], tab);
                            }
                        } else {
#pragma unroll
                            for (int i = 0; i < Q; ++i) {
                                if constexpr (ES == 4) *reinterpret_cast<float *>(o + i * SH::OPITCH + 4) = f[i];
                                else *reinterpret_cast<unsigned short *>(o + i * SH::OPITCH + 2) = (unsigned short)PC::enc1(f[i], tab);
                            }
                        }
                    }
                } else if (fp < pairs) {
                    float f0[Q], f1[Q];
                    unsigned wd[Q];
                    full_mode = pull_cell<Q, F, ALT, 0>(stage + own_b, stage + left_b, stage + right_b, f0, wd, warp_full);
                    full_mode |= pull_cell<Q, F, ALT, 1>(stage + own_b, stage + left_b, stage + right_b, f1, wd, warp_full);
                    collide<COLL, Q, FORCE, SC, ES == 2 ? 1 : 2>(f0, p);  // the shared division (div3)
                    collide<COLL, Q, FORCE, SC, ES == 2 ? 1 : 2>(f1, p);
                    char *o = ostage + 2 * fp * ES;
                    if constexpr (PC::FAST) {
                        // the table-free encoder (P16_0S below 2^-7: every DDF of a flow at LBM velocities); should a value
                        // fall outside its domain, the pair's words are encoded again with the table
                        // (a thread whose inputs needed the full-range decoder goes to the table directly: its results are
                        // of the same size)
                        unsigned acc = full_mode ? PC::FAST_BAD : 0u;
                        if (!full_mode) {
#pragma unroll
                            for (int i = 0; i < Q; ++i) *reinterpret_cast<unsigned *>(o + i * SH::OPITCH) = PC::enc2_fast(f0[i], f1[i], acc);
                        }
                        if (acc & PC::FAST_BAD) {
#pragma unroll
                            for (int i = 0; i < Q; ++i) *reinterpret_cast<unsigned *>(o + i * SH::OPITCH) = PC::enc2(f0[i], f1[i], tab);
                        }
                    } else {
#pragma unroll
                        for (int i = 0; i < Q; ++i) {
                            if constexpr (ES == 4) *reinterpret_cast<float2 *>(o + i * SH::OPITCH) = make_float2(f0[i], f1[i]);
                            else *reinterpret_cast<unsigned *>(o + i * SH::OPITCH) = PC::enc2(f0[i], f1[i], tab);
                        }
                    }
                }
            }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive_n(bar_in_empty + si * 8, SH::CPC);   // once every chunk id has: the input stage may be refilled
            fence_async_smem();                                             // this thread's writes -> visible to the bulk-copy engine
            __syncwarp();
            if (lane == 0) mbar_arrive_n(bar_out_full + so * 8, SH::CPC);
        }
        // The list pass.  The lists of LG consecutive tiles of this CTA (a group; the last one may be shorter) are walked
        // together, LAG tiles after the group's last tile was computed, when its bulk store is complete (`done`; stores
        // complete in order).  A box whose every row ends in a wall has a dozen flagged cells per tile: alone they would
        // occupy a warp -- a third of its lanes -- for a trip to memory and one collision per tile; together they fill the
        // lanes.  The chunk ids of the tile that triggers the pass split the concatenated lists evenly, one cell per lane.
        if (lists && k >= LAG) {
            const int jhi = k - LAG;
            if (jhi % SH::LG == SH::LG - 1 || jhi == my_tiles - 1) {
                const int jlo = jhi - jhi % SH::LG;
                // The headers of the group must be there before they are read.  A chunk of a real tile k has waited for
                // `full` of tile k, which the loader signals after it wrote header k, hence after the headers of all earlier
                // tiles.  A chunk id of one of the LAG trailing pseudo-tiles has waited for nothing: a warp that runs ahead
                // of a lagging loader (FP32 boxes: the kernel waits for memory) would read the ring slot's previous
                // content -- some other tile's list bounds.  `done` of tile jhi implies the header (header -> full ->
                // computed -> stored -> done), so these chunks wait for it first.
                if (k >= my_tiles) mbar_wait(bar_done + (jhi % SH::DONES) * 8, (unsigned)(jhi / SH::DONES) & 1u);
                unsigned lo[SH::LG], end[SH::LG], total = 0;                 // end[g] = lists jlo .. jlo + g, concatenated
#pragma unroll
                for (int gi = 0; gi < SH::LG; ++gi) {
                    lo[gi] = 0;
                    if (jlo + gi <= jhi) {
                        const uint4 hdr = *reinterpret_cast<const uint4 *>(smem + SH::HDR_OFF + ((jlo + gi) % SH::HDRS) * 16);
                        lo[gi] = hdr.y;
                        total += hdr.z - hdr.y;
                    }
                    end[gi] = total;
                }
                if (total != 0) {
                    // (one share per claim of CPC chunk ids: 2^shift / CPC shares)
                    constexpr int CS = SH::CPC == 2 ? 1 : 0;
                    const unsigned share = (((total + (1u << (shift - CS)) - 1u) >> (shift - CS)) + 31u) & ~31u;
                    const unsigned a = (unsigned)(c0 >> CS) * share, b = min(total, a + share);
                    if (a < b) {
                        mbar_wait(bar_done + (jhi % SH::DONES) * 8, (unsigned)(jhi / SH::DONES) & 1u);
                        fence_async_global();
#pragma unroll 1
                        for (unsigned v = a + lane; v < b; v += 32) {
                            int gi = 0;
                            unsigned first = 0;
#pragma unroll
                            for (int q = 0; q + 1 < SH::LG; ++q)
                                if (v >= end[q]) { gi = q + 1; first = end[q]; }
                            unsigned l = lo[0];
#pragma unroll
                            for (int q = 1; q < SH::LG; ++q)
                                if (gi == q) l = lo[q];
                            const uint2 e = __ldg(p.fix_cells + l + (v - first));
                            fix_list_entry<Q, F, FORCE, COLL>(A, B, p, g, (int)blockIdx.x + (jlo + gi) * stride, e);
                        }
                    }
                }
            }
        }
    }
}

}  // namespace lbmk
