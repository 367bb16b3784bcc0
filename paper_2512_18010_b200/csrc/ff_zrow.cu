// ff_zrow.cu — S4 on a Cartesian product grid whose z axis is antisymmetric (z[i] == -z[n-1-i] bit for bit): the row kernel of
// ff_row.cu with a lane's two points chosen as a MIRROR PAIR (+z, -z) of its row (Eq. (45)-(46), (48)
// PAPER.md:309-330).
//
// With g = X Y Z, Z(+-z) = c +- i s, and the polynomial split by the parity of the power of q_z,
//   A + iB at +-z = Pe +- Po,   Pe = sum_{v even} (Ge_v + i Go_v) z^v,   Po = sum_{v odd} (Ge_v + i Go_v) z^v      (ff_row.cu),
// the half sum and half difference of the two points' terms are
//   S' = (f+ + f-)/2 = c E + i (s z) O',    D' = (f+ - f-)/2 = i s E + (c z) O',
//   E = sum_{v even} H_v z^v,   O' = sum_{v odd} H_v z^(v-1),   H_v = X Y (Ge_v + i Go_v)   (warp-uniform: pre-pass).
// A lane accumulates S' and D' — eight FMAs per state for the pair, as before — but E and O' are polynomials in z^2 of half the
// degree, shared by both points, X Y is folded into the H of the pre-pass, and the factor needs no complex product at all (c, s
// from the table, c z and s z): FP64 slots per (q, pair, state) 2 / 4 / 5 / 6 for L = 0..3 (ff_row.cu: 2 / 5 / 7 / 9) and 1-2 per
// (q, pair) (ff_row.cu: 4).  After class 3 the lane converts (S', D') to (f+, f-) = (S' + D', S' - D'); classes L >= 4 run the
// degree blocks of ff_common.cuh on the two points as the other kernels do.  L = 0 needs no pre-pass: S' += (c X Y) D_s,
// D' += (i s X Y) D_s with the four products c a, c b, s a, s b formed once per record.
//
// A warp owns one (ix, iy) row and 32 mirror pairs (lane l: iz = 32 zb + l and nz - 1 - iz); a CTA = 4 consecutive iy.  The Z table
// covers the first half of the axis only (32 complex numbers per record and pair box).  Everything else — the TMA stage ring,
// stream chunks with ordered fix-up tickets, the conjugate store for the inversion mirror, the q-adaptive prefix — as in ff_row.cu.
//
// For state tiles of 4, 8 or 12 states the accumulates of classes 0, 1 and 2 are issued as FP64 tensor-core matrix products over the
// records of a stage (mma.sync.m8n8k4.f64; "classes L = 0..3 on the FP64 tensor cores" below).
#include "ff_common.cuh"

namespace scarf {

namespace {

constexpr int kThreads = 128;
constexpr int kWarps = kThreads / 32;
constexpr int kStages = 2;
constexpr int kStageBytes = 12288;            // records of one stage (>= the largest record, L = 6, NS = 12)
constexpr int kMaxRec = 24;                   // records per stage at most (bounds the table slices)
constexpr int kXB = kZrowBX * 16, kYB = kZrowBY * 16, kZB = kZrowBZ * 16;   // table bytes per record and box
constexpr int kSlotBytes = kStageBytes + kMaxRec * (kXB + kYB + kZB);
static_assert(kMaxRec <= 32 && kZrowBX == 1 && kZrowBY == kWarps && kZrowBZ == 32 && kNQ == 2, "warp = one (ix, iy) row, 32 mirror pairs");

// (parity of n, power of q_z) groups of class L, par 0 first, v ascending (as in ff_row.cu)
__host__ __device__ constexpr bool zgroup_exists(int L, int par, int v) { return ((v & 1) == par ? v : v + 1) <= L; }
__host__ __device__ constexpr int zgroup_index(int L, int par, int v)
{
    int idx = 0;
    for (int p = 0; p < 2; ++p)
        for (int vv = 0; vv <= L; ++vv) {
            if (p == par && vv == v) return idx;
            if (zgroup_exists(L, p, vv)) ++idx;
        }
    return idx;
}
__host__ __device__ constexpr int zgroup_count(int L) { return zgroup_index(L, 2, 0); }
__host__ __device__ constexpr bool zgroup_first(int h)
{
    for (int g = 0; g < h; ++g)
        if (((hdeg(g) ^ hdeg(h)) & 1) == 0 && hexp(g, 2) == hexp(h, 2)) return false;
    return true;
}
__host__ __device__ constexpr int stage_records(int L, int NS)
{
    const int n = kStageBytes / (rec_doubles(L, NS) * 8);
    return n < kMaxRec ? n : kMaxRec;
}
// warp-private area: XY[kMaxRec] (complex; classes 0 and >= 4) followed by H[record][state][v] (complex; classes 1..3)
__host__ __device__ constexpr int h_warp_bytes(int NS)
{
    int m = 16;
    for (int L = 1; L <= 3; ++L) {
        const int b = stage_records(L, NS) * NS * (L + 1) * 16;
        if (b > m) m = b;
    }
    return m + kMaxRec * 16;
}
template <int NS> constexpr int smem_bytes() { return kStages * kSlotBytes + kWarps * h_warp_bytes(NS) + 64; }

// classes kZrowMmaMinL..kZrowMmaMaxL through mma.sync (zrow_mma) for state tiles that fill whole N tiles; the DFMA loops otherwise.
// Measured on config 3 (kernel, ms): no class 5.43; L = 1: 5.10; L = 1..2: 5.00; L = 1..3: 5.00; class 0 besides (zrow_mma0): 4.89; see
// DESIGN.md section 8.
constexpr int kZrowMmaMinL = 1, kZrowMmaMaxL = 2;
template <int L, int NS> constexpr bool kZrowMma = NS % 4 == 0 && L >= kZrowMmaMinL && L <= kZrowMmaMaxL;
// class 0 through mma.sync with its B rows from a per-record table {a, b, -b, a} (zrow_mma0)
template <int NS> constexpr bool kZrowMma0 = NS % 4 == 0;

struct ZPipe {
    unsigned char* buf;     // kStages slots of kSlotBytes: records | X slice | Y slice | Z slice (first half of the axis)
    uint64_t* full;
    uint32_t it;
};

__device__ __forceinline__ double2 cmul(const double2 a, const double2 b)
{
    return make_double2(fma(a.x, b.x, -(a.y * b.y)), fma(a.x, b.y, a.y * b.x));
}

// ---- classes L = 0..3 on the FP64 tensor cores ---------------------------------------------------------------------------------
// The polynomials E = sum_{v even} H_v z^v and z O' = sum_{v odd} H_v z^v have warp-uniform coefficients H_v (pre-pass), so the
// accumulate over the records k of a stage is a real matrix product over (k, v):
//   S'[p][(s, re|im)] += A_S[p][(k, v)] B_S[(k, v)][(s, re|im)],   A_S = c z^v (v even) | s z^v (v odd),   B_S = H_v | i H_v
//   D'[p][(s, re|im)] += A_D[p][(k, v)] B_D[(k, v)][(s, re|im)],   A_D = s z^v (v even) | c z^v (v odd),   B_D = i H_v | H_v
// (p = the warp's 32 mirror pairs).  mma.sync.m8n8k4.f64: four M tiles of eight pairs, N tiles of four states; lane (g, t) =
// (lane / 4, lane % 4) holds A[g][t], B[t][g], C[g][2t, 2t + 1] = (re, im) of pair 8 mt + g and state 4 nt + t.  L + 1 rows per
// record and product: 4 / 8 / 12 / 16 FMAs per mirror pair and state for L = 0..3 (the DFMA loops: 4 / 8 / 10 / 12), but the H of a
// k-tile is read once per warp instead of broadcast to every lane for every state (the DFMA loops of L >= 1 are bound by the
// shared-memory pipe: two wavefronts per broadcast LDS.128, 52 / 76 / 100 per record and warp against 96 / 120 / 144 DFMAs).
// DMMA is counted on the tensor pipe and DFMA on the FP64 pipe, but the two share the FP64 units (64 FMA/clk/SM together): splitting
// the states of a record between a DMMA and a DFMA part in one loop body was slower than either.
__device__ __forceinline__ void dmma884(double (&d)[2], double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d[0]), "+d"(d[1]) : "d"(a), "d"(b));
}
__device__ __forceinline__ double flip_sign(double x, int mask) { return __hiloint2double(__double2hiint(x) ^ mask, __double2loint(x)); }
constexpr int kFragStride(int NS) { return 2 * NS + 2; }   // doubles per pair row of the layout exchange (conflict-free 16-byte accesses)

// per-lane sums (re[h][s], im[h][s]) of pair `lane` <-> C fragments, through the warp's private area (one half h at a time)
template <int NS>
__device__ __forceinline__ void zrow_to_frag(double* W, int lane, const double (&re)[kNQ][NS], const double (&im)[kNQ][NS],
                                             double (&C)[2][4][NS / 4][2])
{
    constexpr int ST = kFragStride(NS);
    static_assert(32 * ST * 8 <= h_warp_bytes(NS), "layout exchange larger than the warp's private area");
    const int g = lane >> 2, t = lane & 3;
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        __syncwarp();
#pragma unroll
        for (int s = 0; s < NS; ++s) *reinterpret_cast<double2*>(W + lane * ST + 2 * s) = make_double2(re[h][s], im[h][s]);
        __syncwarp();
#pragma unroll
        for (int mt = 0; mt < 4; ++mt)
#pragma unroll
            for (int nt = 0; nt < NS / 4; ++nt) {
                const double2 v = *reinterpret_cast<const double2*>(W + (8 * mt + g) * ST + 2 * (4 * nt + t));
                C[h][mt][nt][0] = v.x;
                C[h][mt][nt][1] = v.y;
            }
    }
    __syncwarp();
}
template <int NS>
__device__ __forceinline__ void zrow_from_frag(double* W, int lane, const double (&C)[2][4][NS / 4][2], double (&re)[kNQ][NS],
                                               double (&im)[kNQ][NS])
{
    constexpr int ST = kFragStride(NS);
    const int g = lane >> 2, t = lane & 3;
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        __syncwarp();
#pragma unroll
        for (int mt = 0; mt < 4; ++mt)
#pragma unroll
            for (int nt = 0; nt < NS / 4; ++nt)
                *reinterpret_cast<double2*>(W + (8 * mt + g) * ST + 2 * (4 * nt + t)) = make_double2(C[h][mt][nt][0], C[h][mt][nt][1]);
        __syncwarp();
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            const double2 v = *reinterpret_cast<const double2*>(W + lane * ST + 2 * s);
            re[h][s] = v.x;
            im[h][s] = v.y;
        }
    }
    __syncwarp();
}

// What a lane holds of the A and B fragments does not change along a segment: row rho = 4 j + t of the j-th k-tile of a period
// is term v = rho % (L + 1) (the power of z, the index of H) of record rho / (L + 1) of the period's records.
//   v even:  S' column c z^v with row H_v,    D' column s z^v with row i H_v
//   v odd:   S' column s z^v with row i H_v,  D' column c z^v with row H_v          (i H = (-H_i, H_r))
template <int L>
struct ZMmaLane {
    static constexpr int NV = L + 1;
    static constexpr int P = NV == 3 ? 3 : 1;             // k-tiles per period (4 P rows = R records of NV rows)
    static constexpr int R = 4 * P / NV;
    static_assert(4 * P == R * NV, "a period holds whole records");
    int zoff[P];        // doubles from (c, s)[first record of the period][pair 8 mt + g] to this lane's S' factor (the D' factor: ^ 1)
    int odd[P];         // v & 1
    int hoff[P];        // doubles from H[first record][state 4 nt][0] to this lane's H_v of state 4 nt + g / 2
    int drec[P];        // record of the period
    int o1[P];          // component of H_v the S' row holds (the D' row: the other)
    int neg1[P], neg2[P];   // sign-bit masks of the S' / D' row
    double sc[P][4];    // z^v of pair 8 mt + g
};
template <int L, int NS>
__device__ __forceinline__ void zrow_mma_lane(double z, int lane, ZMmaLane<L>& m)
{
    constexpr int NV = L + 1;
    const int g = lane >> 2, t = lane & 3, comp = g & 1;
    double zq[4];
#pragma unroll
    for (int mt = 0; mt < 4; ++mt) zq[mt] = __shfl_sync(0xffffffffu, z, 8 * mt + g);
#pragma unroll
    for (int j = 0; j < ZMmaLane<L>::P; ++j) {
        const int rho = 4 * j + t, v = rho % NV, dr = rho / NV, ty = v & 1;
        m.drec[j] = dr;
        m.odd[j] = ty;
        m.zoff[j] = dr * kZrowBZ * 2 + g * 2 + ty;
        m.hoff[j] = ((dr * NS + (g >> 1)) * NV + v) * 2;
        m.o1[j] = ty ? 1 - comp : comp;
        m.neg1[j] = (ty == 1 && comp == 0) ? (int)0x80000000 : 0;
        m.neg2[j] = (ty == 0 && comp == 0) ? (int)0x80000000 : 0;
#pragma unroll
        for (int mt = 0; mt < 4; ++mt) {
            double p = 1.0;
#pragma unroll
            for (int e = 1; e <= L; ++e)
                if (e <= v) p *= zq[mt];
            m.sc[j][mt] = p;
        }
    }
}

// the records of one stage: Hd = the pre-pass' H[record][state][v] (complex) as doubles, Zd = the stage's Z slice (c, s)[record][pair]
// as doubles
template <int L, int NS>
__device__ __forceinline__ void zrow_mma(const double* __restrict__ Hd, const double* __restrict__ Zd, int cnt, const ZMmaLane<L>& m,
                                         double (&C)[2][4][NS / 4][2])
{
    constexpr int NT = NS / 4, NV = L + 1, P = ZMmaLane<L>::P, R = ZMmaLane<L>::R;
#pragma unroll(P == 1 ? 2 : 1)
    for (int k0 = 0; k0 < cnt; k0 += R) {
        const double* zb = Zd + k0 * kZrowBZ * 2;
        const double* hb = Hd + k0 * NS * NV * 2;
#pragma unroll
        for (int j = 0; j < P; ++j) {
            const bool valid = k0 + m.drec[j] < cnt;      // a short last period: the rows of the missing records are zero
            double a1[4], a2[4], b1[NT], b2[NT];
#pragma unroll
            for (int mt = 0; mt < 4; ++mt) {
                const double* zp = zb + m.zoff[j] + 16 * mt;
                const double u = valid ? zp[0] : 0.0, v = valid ? zp[1 - 2 * m.odd[j]] : 0.0;
                a1[mt] = u * m.sc[j][mt];                   // c z^v | s z^v
                a2[mt] = v * m.sc[j][mt];                   // s z^v | c z^v
            }
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) {
                const double* hp = hb + m.hoff[j] + 4 * nt * NV * 2;
                b1[nt] = flip_sign(valid ? hp[m.o1[j]] : 0.0, m.neg1[j]);
                b2[nt] = flip_sign(valid ? hp[1 - m.o1[j]] : 0.0, m.neg2[j]);
            }
#pragma unroll
            for (int mt = 0; mt < 4; ++mt)
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                    dmma884(C[0][mt][nt], a1[mt], b1[nt]);
                    dmma884(C[1][mt][nt], a2[mt], b2[nt]);
                }
        }
    }
}

// ---- class 0 on the tensor cores: S' += c (X Y D_s), D' += s (i X Y D_s).  A k-tile = four records, one row each.  pq[record] =
// {a, b, -b, a} with X Y = a + i b (written by lane `record` before the loop): the S' row of lane (g, t) is pq[g & 1] D_s, the D' row
// pq[2 + (g & 1)] D_s, for record k0 + t and state 4 nt + g / 2; the A columns are c and s as they stand in the Z slice.
template <int NS>
__device__ __forceinline__ void zrow_mma0(const unsigned char* __restrict__ sp, const double* __restrict__ pq, const double* __restrict__ Zd,
                                          int cnt, int lane, double (&C)[2][4][NS / 4][2])
{
    constexpr int NT = NS / 4, REC = rec_doubles(0, NS) * 8;
    const int g = lane >> 2, t = lane & 3, comp = g & 1;
#pragma unroll 2
    for (int k0 = 0; k0 < cnt; k0 += 4) {
        const bool valid = k0 + t < cnt;                    // a short last k-tile: the B rows of the missing records are zero
        const int r = valid ? k0 + t : k0;                  // (their A columns: those of a record that exists, finite)
        const double p = valid ? pq[r * 4 + comp] : 0.0, q = valid ? pq[r * 4 + 2 + comp] : 0.0;
        const double* D = reinterpret_cast<const double*>(sp + r * REC) + 4 + (g >> 1);
        double a1[4], a2[4], b1[NT], b2[NT];
#pragma unroll
        for (int mt = 0; mt < 4; ++mt) {
            const double2 zc = *reinterpret_cast<const double2*>(Zd + (r * kZrowBZ + 8 * mt + g) * 2);
            a1[mt] = zc.x;
            a2[mt] = zc.y;
        }
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
            const double d = D[4 * nt];
            b1[nt] = p * d;
            b2[nt] = q * d;
        }
#pragma unroll
        for (int mt = 0; mt < 4; ++mt)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) {
                dmma884(C[0][mt][nt], a1[mt], b1[nt]);
                dmma884(C[1][mt][nt], a2[mt], b2[nt]);
            }
    }
}

// ---- pre-pass: H[record][state][v] = X Y (Ge_v + i Go_v) of one stage for this warp's row --------------------------------------
// xym[yz_index(t, u)] = q_x^t q_y^u (1 <= t + u <= L).  One (record, state) pair per lane and trip.
template <int L, int NS>
__device__ __forceinline__ void zrow_prepass(const unsigned char* sp, int cnt, const double2* Xs, const double2* Ys,
                                             const double (&xym)[yz_count(L)], double2* Hw, int lane)
{
    constexpr int REC = rec_doubles(L, NS) * 8, NH = nherm(L), NG = zgroup_count(L);
    constexpr int TRIPS = (stage_records(L, NS) * NS + 31) / 32;
    const int n = cnt * NS;
#pragma unroll 5
    for (int tr = 0; tr < TRIPS; ++tr) {
        const int i = lane + 32 * tr;
        if (i >= n) break;
        const int k = i / NS, s = i - k * NS;
        const double* D = reinterpret_cast<const double*>(sp + k * REC) + 4 + s * NH;
        const double2 xy = cmul(Xs[k * kZrowBX], Ys[k * kZrowBY]);
        double G[NG];
        static_for<NH>([&](auto hc) {
            constexpr int h = decltype(hc)::value;
            constexpr int t = hexp(h, 0), u = hexp(h, 1), v = hexp(h, 2), g = zgroup_index(L, hdeg(h) & 1, v);
            const double cv = D[h];
            if constexpr (t + u == 0) G[g] = cv;
            else if constexpr (zgroup_first(h)) G[g] = cv * xym[yz_index(t, u)];
            else G[g] = fma(cv, xym[yz_index(t, u)], G[g]);
        });
        double2* o = Hw + (size_t)(k * NS + s) * (L + 1);
        static_for<L + 1>([&](auto vc) {
            constexpr int v = decltype(vc)::value;
            constexpr bool he = zgroup_exists(L, 0, v), ho = zgroup_exists(L, 1, v);
            double2 H;
            if constexpr (he && ho) {
                const double ge = G[zgroup_index(L, 0, v)], go = G[zgroup_index(L, 1, v)];
                H = make_double2(fma(xy.x, ge, -(xy.y * go)), fma(xy.x, go, xy.y * ge));
            } else if constexpr (he) {
                const double ge = G[zgroup_index(L, 0, v)];
                H = make_double2(xy.x * ge, xy.y * ge);
            } else {
                const double go = G[zgroup_index(L, 1, v)];
                H = make_double2(-(xy.y * go), xy.x * go);
            }
            o[v] = H;
        });
    }
}

// ---- one record, L = 1..3: S' += c E + i (s z) O',  D' += i s E + (c z) O'  (re[0], im[0] = S'; re[1], im[1] = D') --------------
// zf = {c, s, c z, s z} of this lane's pair; z2 = z^2.
template <int L, int NS>
__device__ __forceinline__ void record_accum_zrow(const double2* __restrict__ H, const double (&zf)[4], double z2,
                                                  double (&re)[kNQ][NS], double (&im)[kNQ][NS])
{
    static_for<NS>([&](auto sc) {
        constexpr int s = decltype(sc)::value;
        const double2 h0 = H[s * (L + 1)], h1 = H[s * (L + 1) + 1];
        double Er = h0.x, Ei = h0.y, Or = h1.x, Oi = h1.y;
        if constexpr (L >= 2) {
            const double2 h2 = H[s * (L + 1) + 2];
            Er = fma(h2.x, z2, Er);
            Ei = fma(h2.y, z2, Ei);
        }
        if constexpr (L >= 3) {
            const double2 h3 = H[s * (L + 1) + 3];
            Or = fma(h3.x, z2, Or);
            Oi = fma(h3.y, z2, Oi);
        }
        re[0][s] = fma(zf[0], Er, re[0][s]);
        re[0][s] = fma(-zf[3], Oi, re[0][s]);
        im[0][s] = fma(zf[0], Ei, im[0][s]);
        im[0][s] = fma(zf[3], Or, im[0][s]);
        re[1][s] = fma(-zf[1], Ei, re[1][s]);
        re[1][s] = fma(zf[2], Or, re[1][s]);
        im[1][s] = fma(zf[1], Er, im[1][s]);
        im[1][s] = fma(zf[2], Oi, im[1][s]);
    });
}

// ---- one class segment of the chunk ----------------------------------------------------------------------------------------
// r0 = stream-order index of the segment's first record (row of the tables).  qv[0] = (q_x, q_y, +z, 0), qv[1] = (q_x, q_y, -z, 0).
// Classes 0..3 accumulate (S', D') in (re[0], im[0]), (re[1], im[1]); classes >= 4 the two points' own sums (converted in between).
template <int L, int NS>
__device__ __forceinline__ void run_class_zrow(ZPipe& pp, const GridArgs& a, const char* __restrict__ seg, long long r0, int n_rec,
                                               int bx, int by, int bz, int warp, int lane, double* Ww,
                                               const double (&qv)[kNQ][4], double (&re)[kNQ][NS], double (&im)[kNQ][NS])
{
    constexpr int REC = rec_doubles(L, NS) * 8;
    constexpr int SREC = stage_records(L, NS);
    static_assert(SREC >= 1, "record larger than a stage");
    const int n_st = (n_rec + SREC - 1) / SREC;
    const bool producer = threadIdx.x == 0;
    auto issue = [&](int j) {
        const int slot = (int)((pp.it + (uint32_t)j) % kStages);
        const int first = j * SREC, cnt = min(SREC, n_rec - first);
        unsigned char* sb = pp.buf + slot * kSlotBytes;
        const long long r = r0 + first;
        SCARF_CHECK(cnt >= 1 && cnt <= kMaxRec && cnt * REC <= kStageBytes && r >= 0 && r + cnt <= a.n_rows && slot >= 0 && slot < kStages);
        mbar_expect_tx(&pp.full[slot], (uint32_t)cnt * (REC + kXB + kYB + kZB));
        bulk_g2s(sb, seg + (size_t)first * REC, (uint32_t)cnt * REC, &pp.full[slot]);
        bulk_g2s(sb + kStageBytes, a.tx + ((size_t)bx * a.n_rows + r) * kZrowBX, (uint32_t)cnt * kXB, &pp.full[slot]);
        bulk_g2s(sb + kStageBytes + kMaxRec * kXB, a.ty + ((size_t)by * a.n_rows + r) * kZrowBY, (uint32_t)cnt * kYB, &pp.full[slot]);
        bulk_g2s(sb + kStageBytes + kMaxRec * (kXB + kYB), a.tz + ((size_t)bz * a.n_rows + r) * kZrowBZ, (uint32_t)cnt * kZB,
                 &pp.full[slot]);
    };
    const double z = qv[0][2], z2 = z * z;
    double xym[(L >= 1 && L <= 3) ? yz_count(L) : 1];
    if constexpr (L >= 1 && L <= 3) {
        double pv[kNQ][4], zp_unused[kNQ][L + 1];
#pragma unroll
        for (int j = 0; j < kNQ; ++j) { pv[j][0] = 0.0; pv[j][1] = qv[0][0]; pv[j][2] = qv[0][1]; pv[j][3] = 0.0; }
        make_xpair_monomials<L>(pv, xym, zp_unused);      // xym[yz_index(t, u)] = q_x^t q_y^u
    }
    __syncthreads();                                     // all threads have left the previous segment's stages
    if (producer)
        for (int j = 0; j < min(kStages, n_st); ++j) issue(j);
    // L = 1 on the tensor cores: the sums live in C fragments for the length of the segment
    constexpr bool MMA0 = L == 0 && kZrowMma0<NS>, MMA = kZrowMma<L, NS>;
    double Cf[2][4][(MMA || MMA0) ? NS / 4 : 1][2];
    ZMmaLane<MMA ? L : 1> ml;
    if constexpr (MMA) zrow_mma_lane<L, NS>(z, lane, ml);
    if constexpr (MMA || MMA0) zrow_to_frag<NS>(Ww, lane, re, im, Cf);
    for (int j = 0; j < n_st; ++j) {
        const uint32_t g = pp.it + (uint32_t)j;
        const int slot = (int)(g % kStages);
        mbar_wait(&pp.full[slot], (g / kStages) & 1u);
        const int cnt = min(SREC, n_rec - j * SREC);
        const unsigned char* sp = pp.buf + slot * kSlotBytes;
        const double2* Xs = reinterpret_cast<const double2*>(sp + kStageBytes);
        const double2* Ys = reinterpret_cast<const double2*>(sp + kStageBytes + kMaxRec * kXB) + warp;
        const double2* Zs = reinterpret_cast<const double2*>(sp + kStageBytes + kMaxRec * (kXB + kYB)) + lane;
        double2* XYw = reinterpret_cast<double2*>(Ww);
        double2* Hw = XYw + kMaxRec;
        if constexpr (MMA0) {
            double* pq = reinterpret_cast<double*>(Hw);
            if (lane < cnt) {
                const double2 xy = cmul(Xs[lane * kZrowBX], Ys[lane * kZrowBY]);
                *reinterpret_cast<double2*>(pq + lane * 4) = xy;
                *reinterpret_cast<double2*>(pq + lane * 4 + 2) = make_double2(-xy.y, xy.x);
            }
            __syncwarp();
            zrow_mma0<NS>(sp, pq, reinterpret_cast<const double*>(sp + kStageBytes + kMaxRec * (kXB + kYB)), cnt, lane, Cf);
        } else if constexpr (MMA) {
            zrow_prepass<L, NS>(sp, cnt, Xs, Ys, xym, Hw, lane);
            __syncwarp();
            zrow_mma<L, NS>(reinterpret_cast<const double*>(Hw), reinterpret_cast<const double*>(sp + kStageBytes + kMaxRec * (kXB + kYB)),
                            cnt, ml, Cf);
        } else if constexpr (L >= 1 && L <= 3) {
            zrow_prepass<L, NS>(sp, cnt, Xs, Ys, xym, Hw, lane);
            __syncwarp();
            // {c, s, c z, s z} of record k; software-pipelined by groups of U records
            auto factors = [&](int k, double (&zf)[4]) {
                const double2 Zk = Zs[k * kZrowBZ];
                zf[0] = Zk.x; zf[1] = Zk.y; zf[2] = Zk.x * z; zf[3] = Zk.y * z;
            };
            constexpr int U = L <= 1 ? 2 : 1;
            const int n_full = cnt / U * U;
            double zf[U][4];
            if (n_full > 0) {
#pragma unroll
                for (int u = 0; u < U; ++u) factors(u, zf[u]);
#pragma unroll 1
                for (int k = 0; k + U < n_full; k += U) {
                    double zn[U][4];
#pragma unroll
                    for (int u = 0; u < U; ++u) factors(k + U + u, zn[u]);
#pragma unroll
                    for (int u = 0; u < U; ++u) record_accum_zrow<L, NS>(Hw + (size_t)(k + u) * NS * (L + 1), zf[u], z2, re, im);
#pragma unroll
                    for (int u = 0; u < U; ++u)
#pragma unroll
                        for (int c = 0; c < 4; ++c) zf[u][c] = zn[u][c];
                }
#pragma unroll
                for (int u = 0; u < U; ++u) record_accum_zrow<L, NS>(Hw + (size_t)(n_full - U + u) * NS * (L + 1), zf[u], z2, re, im);
            }
#pragma unroll 1
            for (int k = n_full; k < cnt; ++k) {
                factors(k, zf[0]);
                record_accum_zrow<L, NS>(Hw + (size_t)k * NS * (L + 1), zf[0], z2, re, im);
            }
        } else {
            // X Y of the row, once per record (lane k: record k)
            if (lane < cnt) XYw[lane] = cmul(Xs[lane * kZrowBX], Ys[lane * kZrowBY]);
            __syncwarp();
            if constexpr (L == 0) {
                // S' += (c X Y) D_s, D' += (i s X Y) D_s: the accumulate of the other kernels with gc = {c a, -s b}, gs = {c b, s a}
                auto factors = [&](int k, double (&gc)[kNQ], double (&gs)[kNQ]) {
                    const double2 xy = XYw[k], Zk = Zs[k * kZrowBZ];
                    gc[0] = Zk.x * xy.x; gs[0] = Zk.x * xy.y;
                    gc[1] = -(Zk.y * xy.y); gs[1] = Zk.y * xy.x;
                };
                auto accum = [&](int k, const double (&gc)[kNQ], const double (&gs)[kNQ]) {
                    double mono[kNQ][1];
#pragma unroll
                    for (int jj = 0; jj < kNQ; ++jj) mono[jj][0] = 1.0;
                    record_accum<0, NS, kNQ, 0>(reinterpret_cast<const double2*>(sp + k * REC), mono, gc, gs, re, im);
                };
                constexpr int U = 2;
                const int n_full = cnt / U * U;
                double gc[U][kNQ], gs[U][kNQ];
                if (n_full > 0) {
#pragma unroll
                    for (int u = 0; u < U; ++u) factors(u, gc[u], gs[u]);
#pragma unroll 1
                    for (int k = 0; k + U < n_full; k += U) {
                        double gcn[U][kNQ], gsn[U][kNQ];
#pragma unroll
                        for (int u = 0; u < U; ++u) factors(k + U + u, gcn[u], gsn[u]);
#pragma unroll
                        for (int u = 0; u < U; ++u) accum(k + u, gc[u], gs[u]);
#pragma unroll
                        for (int u = 0; u < U; ++u)
#pragma unroll
                            for (int jj = 0; jj < kNQ; ++jj) { gc[u][jj] = gcn[u][jj]; gs[u][jj] = gsn[u][jj]; }
                    }
#pragma unroll
                    for (int u = 0; u < U; ++u) accum(n_full - U + u, gc[u], gs[u]);
                }
#pragma unroll 1
                for (int k = n_full; k < cnt; ++k) {
                    factors(k, gc[0], gs[0]);
                    accum(k, gc[0], gs[0]);
                }
            } else {                                    // L >= 4: degree blocks on the two points (+z, -z); g = X Y (c +- i s)
#pragma unroll 1
                for (int k0 = 0; k0 < cnt; k0 += kBlkRec) {
                    const int nb = min(kBlkRec, cnt - k0);
                    double gcb[kBlkRec][kNQ], gsb[kBlkRec][kNQ];
                    static_for<kBlkRec>([&](auto rc) {
                        constexpr int r = decltype(rc)::value;
                        if (r < nb) {
                            const double2 xy = XYw[k0 + r], Zk = Zs[(k0 + r) * kZrowBZ];
                            const double2 gp = cmul(xy, Zk), gm = cmul(xy, make_double2(Zk.x, -Zk.y));
                            gcb[r][0] = gp.x; gsb[r][0] = gp.y;
                            gcb[r][1] = gm.x; gsb[r][1] = gm.y;
                        }
                    });
                    accum_blocks<L, NS>(sp + k0 * REC, nb, qv, gcb, gsb, re, im);
                }
            }
        }
        __syncthreads();                                 // the slot and the warp areas are free again
        if (producer && j + kStages < n_st) issue(j + kStages);
    }
    pp.it += (uint32_t)n_st;
    if constexpr (MMA || MMA0) zrow_from_frag<NS>(Ww, lane, Cf, re, im);
}

template <int NS>
__global__ void __launch_bounds__(kThreads, 2) ff_zrow_kernel(const GridArgs a)
{
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem + kStages * kSlotBytes);
    int tile, chunk;
    cta_tile_chunk(a.v, tile, chunk);
    if (threadIdx.x == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(&full_bar[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    ZPipe pp = {smem, full_bar, 0u};
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double* Ww = reinterpret_cast<double*>(smem + kStages * kSlotBytes + 64 + warp * h_warp_bytes(NS));   // the warp's private area

    const int bz = tile % a.nbz, by = (tile / a.nbz) % a.nby, bx = a.bx0 + tile / (a.nbz * a.nby);
    const int ix = bx, iy = by * kZrowBY + warp;
    const int nz_half = (a.nz + 1) / 2;                   // mirror pairs of a row (the middle point of an odd axis pairs with itself)
    const int izp = bz * kZrowBZ + lane, izm = a.nz - 1 - izp;
    const bool row_ok = ix < a.nx_eval && iy < a.ny, ok = row_ok && izp < nz_half;
    double qv[kNQ][4];
#pragma unroll
    for (int j = 0; j < kNQ; ++j) {
        qv[j][0] = row_ok ? a.qx[ix] : 0.0;            // the row's q_x, q_y are warp-uniform whatever iz is
        qv[j][1] = row_ok ? a.qy[iy] : 0.0;
        qv[j][3] = 0.0;
    }
    qv[0][2] = ok ? a.qz[izp] : 0.0;
    qv[1][2] = -qv[0][2];                                // the axis is antisymmetric bit for bit (checked by the host)
    double re[kNQ][NS], im[kNQ][NS];
#pragma unroll
    for (int j = 0; j < kNQ; ++j)
#pragma unroll
        for (int s = 0; s < NS; ++s) re[j][s] = im[j][s] = 0.0;

    __shared__ CtaPlan plan;                                // per class: the records this CTA evaluates; its ticket turn (ff_common.cuh)
    {
        const double m2 = ok ? qv[0][0] * qv[0][0] + qv[0][1] * qv[0][1] + qv[0][2] * qv[0][2] : 1e300;      // |q| of +z and -z agree
        plan_cta<NS>(a.v, chunk, m2, plan);
    }
#define SCARF_ZROW_CLASS(LV)                                                                                         \
    if (plan.nrec[LV] > 0)                                                                                           \
        run_class_zrow<LV, NS>(pp, a, a.v.base + plan.off[LV], plan.row[LV], plan.nrec[LV], bx, by, bz, warp, lane, Ww, qv, re, im);
    SCARF_ZROW_CLASS(0)
    SCARF_ZROW_CLASS(1)
    SCARF_ZROW_CLASS(2)
    SCARF_ZROW_CLASS(3)
    // (S', D') -> (f+, f-) = (S' + D', S' - D')
#pragma unroll
    for (int s = 0; s < NS; ++s) {
        const double sr = re[0][s], si = im[0][s], dr = re[1][s], di = im[1][s];
        re[0][s] = sr + dr; im[0][s] = si + di;
        re[1][s] = sr - dr; im[1][s] = si - di;
    }
    SCARF_ZROW_CLASS(4)
    SCARF_ZROW_CLASS(5)
    SCARF_ZROW_CLASS(6)
#undef SCARF_ZROW_CLASS

    // ---- epilogue: store (one chunk) or add into `out` in chunk order (several); the LAST chunk holds the final value and
    // also stores its conjugate at the inversion-mirror point when the whole grid is inversion-symmetric
    double2* dst = reinterpret_cast<double2*>(a.v.dst);
    double2* fin = a.v.dst_final != nullptr ? reinterpret_cast<double2*>(a.v.dst_final) : dst;    // finished values (last chunk)
    const int turn = plan.turn;
    if (turn < 0) return;                                   // a chunk without work (uniform over the CTA)
    const bool first = turn == 0, last = plan.next == 0;
    if (a.v.n_chunks > 1) ticket_wait(a.v.tickets + tile, turn);
#pragma unroll
    for (int j = 0; j < kNQ; ++j) {
        const int iz = j == 0 ? izp : izm;
        if (ok && (j == 0 || izm != izp)) {                 // the middle point of an odd axis is its own partner: stored once
            const long long i = ((long long)ix * a.ny + iy) * a.nz + iz;
            const bool mirror = last && a.sym && 2 * ix < a.nx - 1;
            SCARF_CHECK(i >= 0 && i < a.v.n_q);
#pragma unroll
            for (int s = 0; s < NS; ++s)
                if (s < a.v.ns_real) {
                    double2* o = dst + (size_t)s * a.v.n_q;
                    double2 v = make_double2(re[j][s], im[j][s]);
                    if (!first) {
                        const double2 p = __ldcg(o + i);
                        v.x += p.x;
                        v.y += p.y;
                    }
                    double2* w = (last ? fin : dst) + (size_t)s * a.v.n_q;
                    w[i] = v;
                    if (mirror) w[a.v.n_q - 1 - i] = make_double2(v.x, -v.y);   // f(-q) = conj f(q)
                }
        }
    }
    if (a.v.n_chunks > 1) ticket_pass(a.v.tickets + tile, plan.next);
}

template <int NS>
cudaError_t launch_zrow_ns(const GridArgs& a, cudaStream_t st)
{
    const dim3 grid((unsigned)a.v.n_tiles, (unsigned)a.v.n_chunks, 1);   // dispatched x fastest: chunk-major
    ff_zrow_kernel<NS><<<grid, kThreads, smem_bytes<NS>(), st>>>(a);
    return cudaGetLastError();
}

}  // namespace

// The kernels need more than 48 KB of dynamic shared memory: an attribute of the function on the CURRENT device.  Called by
// scarf_create for the context's device (idempotent, no process-wide flag).
cudaError_t ff_zrow_init_device()
{
    cudaError_t e = cudaSuccess;
#define SCARF_ZROW_ATTR(NSV) \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(ff_zrow_kernel<NSV>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes<NSV>());
    SCARF_ZROW_ATTR(1) SCARF_ZROW_ATTR(2) SCARF_ZROW_ATTR(4) SCARF_ZROW_ATTR(6) SCARF_ZROW_ATTR(8) SCARF_ZROW_ATTR(12)
#undef SCARF_ZROW_ATTR
    return e;
}

// a.nz is the FULL axis length; a.nbz counts boxes of 32 mirror pairs; the Z table covers the first ceil(nz/2) points
cudaError_t launch_ff_zrow(int NS, const GridArgs& a, cudaStream_t st)
{
    if (a.v.n_q <= 0 || a.v.n_chunks <= 0 || a.v.n_tiles <= 0) return cudaSuccess;
    if (a.bxs != kZrowBX || a.bys != kZrowBY || a.bzs != kZrowBZ) return cudaErrorInvalidValue;   // tables laid out for another kernel
    switch (NS) {
    case 1: return launch_zrow_ns<1>(a, st);
    case 2: return launch_zrow_ns<2>(a, st);
    case 4: return launch_zrow_ns<4>(a, st);
    case 6: return launch_zrow_ns<6>(a, st);
    case 8: return launch_zrow_ns<8>(a, st);
    case 12: return launch_zrow_ns<12>(a, st);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace scarf
