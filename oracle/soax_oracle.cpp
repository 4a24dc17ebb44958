// soax_oracle.cpp -- the ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, single-threaded CPU statement of what the SoAx hot path computes, over an
// ARRAY OF STRUCTS, written from the paper and from BASELINE.json's config text under the
// readings Q1..Q16 of SURVEY.md section 8(c) (listed again in DESIGN.md).  It shares no code, header,
// helper, table or constant with the CUDA path under paper_1710_03462_b200/csrc/ and neither includes the
// other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// load it.  Build: g++ -std=c++17 -O2 -ffp-contract=off -fno-fast-math -shared -fPIC (see oracle/build.py);
// every fused multiply-add below is an explicit std::fma / std::fmaf, nothing else may be contracted.
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): closed-form drift, wrap properties, the exact invariant
// and the linear closed form of the symplectic-Euler map, the exact RK2 energy growth factor, the 4-particle
// dyadic energy fixture, exact rational summation, byte-exact AoS<->SoA round trips against numpy structured
// arrays, the 6-particle binning fixture of SURVEY.md 8(c), O(N^2) brute-force ranks for N <= 64, and
// numpy's stable argsort at larger N; the energy of the wide record (double vel) by the same fixture stored as R2
// and by exact rationals.  No arithmetic function here is "parity unpinned" (the seeded input generator lives in
// paper_1710_03462_b200/inputs.py, is unpinned, and feeds both sides the same arrays).
//
// Records (declaration order, SURVEY.md section 8 "Records used by the configs"):
//   R1  PAPER.md:41  {int32 id; double pos[3]; float vel[3]}  packed, stride 40, offsets 0/4,12,20/28,32,36 (Q1)
//   R2  config 4     {int64 id; double pos[3]; double vel[3]; double acc[3]; float mass; float charge;
//                     uint8 flags}  natural C layout, stride 96
//   B6  PAPER.md:144-153 (Listing 4, SIZE extra floats) {float x[3]; float v[3]; float temp[SIZE]}
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <algorithm>

namespace {

#pragma pack(push, 1)
struct R1 {            // 40 bytes, no padding (Q1): doubles sit at offset 4 mod 8
    int32_t id;
    double  pos[3];
    float   vel[3];
};
#pragma pack(pop)
static_assert(sizeof(R1) == 40, "R1 must be the 40-byte packed record of BASELINE.json config 3");

struct R2 {            // natural alignment: 8 + 72 + 4 + 4 + 1 (+7 pad) = 96
    int64_t id;
    double  pos[3];
    double  vel[3];
    double  acc[3];
    float   mass;
    float   charge;
    uint8_t flags;
};
static_assert(sizeof(R2) == 96, "R2 natural layout");

// Q3: wrap into [0,1):  w = x - floor(x); a result of exactly 1.0 (x = -tiny) maps to 0.0.
inline double wrap(double x) {
    double w = x - std::floor(x);
    if (w >= 1.0) w = 0.0;
    return w;
}

// Packed records: every field goes through memcpy (misaligned doubles).
inline R1 load1(const unsigned char* base, int64_t i) { R1 r; std::memcpy(&r, base + 40 * i, 40); return r; }
inline void store1(unsigned char* base, int64_t i, const R1& r) { std::memcpy(base + 40 * i, &r, 40); }

// Neumaier-compensated running sum (SURVEY.md 8(c) ENERGY: "sum_i e_i in index order with
// Neumaier-compensated double summation").
struct Neumaier {
    double s = 0.0, c = 0.0;
    void add(double x) {
        double t = s + x;
        if (std::fabs(s) >= std::fabs(x)) c += (s - t) + x; else c += (x - t) + s;
        s = t;
    }
    double value() const { return s + c; }
};

// Q16 / a10: i_c = (int32)(pos_c * G) (exact product for G a power of two; truncation), x slowest (Q11).
inline int64_t cell_of(const double p[3], int32_t G) {
    int32_t i0 = (int32_t)(p[0] * (double)G);
    int32_t i1 = (int32_t)(p[1] * (double)G);
    int32_t i2 = (int32_t)(p[2] * (double)G);
    return ((int64_t)i0 * G + i1) * G + i2;
}

}  // namespace

extern "C" {

// ---- a3 ------------------------------------------------------------------------------------------------
double soax_oracle_wrap(double x) { return wrap(x); }

int64_t soax_oracle_r1_stride(void) { return (int64_t)sizeof(R1); }
int64_t soax_oracle_r2_stride(void) { return (int64_t)sizeof(R2); }
// offsets of id, pos[0..2], vel[0..2] in the packed record (Q1), from the compiler, not from a table
void soax_oracle_r1_offsets(int64_t out[7]) {
    R1 r; const char* b = (const char*)&r;
    out[0] = (const char*)&r.id - b;
    for (int c = 0; c < 3; ++c) out[1 + c] = (const char*)&r.pos[c] - b;
    for (int c = 0; c < 3; ++c) out[4 + c] = (const char*)&r.vel[c] - b;
}

// ---- a2: DRIFT (Eq. 1 "x += dt v", with periodic wrap; configs 1, 5) ------------------------
//      pos[c] = wrap( fma(dt, (double)vel[c], pos[c]) ),  one full pass over all particles per step (Q14).
void soax_oracle_r1_drift(void* aos, int64_t n, double dt, int32_t nsteps) {
    unsigned char* base = (unsigned char*)aos;
    for (int32_t s = 0; s < nsteps; ++s)
        for (int64_t i = 0; i < n; ++i) {
            R1 p = load1(base, i);
            for (int c = 0; c < 3; ++c) p.pos[c] = wrap(std::fma(dt, (double)p.vel[c], p.pos[c]));
            store1(base, i, p);
        }
}

// ---- a4: SYMPLECTIC EULER, harmonic, kick then drift with the NEW velocity (Q2, Q4; configs 2, 3) --------
//      F = (float)( -(k * (pos[c] - ctr)) );  vel[c] = fmaf((float)dt, F, vel[c]);
//      pos[c] = wrap( fma(dt, (double)vel[c], pos[c]) ).          (k = 1 in the configs: k*x is then exact)
void soax_oracle_r1_symplectic_euler(void* aos, int64_t n, double dt, double k, double ctr, int32_t nsteps) {
    unsigned char* base = (unsigned char*)aos;
    const float dt_f = (float)dt;
    for (int32_t s = 0; s < nsteps; ++s)
        for (int64_t i = 0; i < n; ++i) {
            R1 p = load1(base, i);
            for (int c = 0; c < 3; ++c) {
                float F = (float)(-(k * (p.pos[c] - ctr)));
                p.vel[c] = std::fmaf(dt_f, F, p.vel[c]);
                p.pos[c] = wrap(std::fma(dt, (double)p.vel[c], p.pos[c]));
            }
            store1(base, i, p);
        }
}

// ---- a9: RK2 MIDPOINT, harmonic force -k (pos-ctr)/mass, masked by flags (config 4; Q6, Q7, Q8) ---------
void soax_oracle_r2_rk2(void* aos, int64_t n, double dt, double k, double ctr, uint8_t mask, int32_t nsteps) {
    R2* P = (R2*)aos;
    const double hh = 0.5 * dt;
    for (int32_t s = 0; s < nsteps; ++s)
        for (int64_t i = 0; i < n; ++i) {
            R2& p = P[i];
            if ((p.flags & mask) == 0) continue;               // no field changes
            const double w = k / (double)p.mass;               // Q8: one IEEE division per particle
            double a1[3], ph[3], vh[3], a2[3];
            for (int c = 0; c < 3; ++c) a1[c] = -(w * (p.pos[c] - ctr));
            for (int c = 0; c < 3; ++c) {
                ph[c] = wrap(std::fma(hh, p.vel[c], p.pos[c]));  // Q6: force is evaluated on the torus
                vh[c] = std::fma(hh, a1[c], p.vel[c]);
            }
            for (int c = 0; c < 3; ++c) a2[c] = -(w * (ph[c] - ctr));
            for (int c = 0; c < 3; ++c) {
                p.pos[c] = wrap(std::fma(dt, vh[c], p.pos[c]));
                p.vel[c] = std::fma(dt, a2[c], p.vel[c]);
                p.acc[c] = a2[c];                               // Q7
            }
        }
}

// DRIFT on the wide record (double vel): same Eq. 1 update.
void soax_oracle_r2_drift(void* aos, int64_t n, double dt, int32_t nsteps) {
    R2* P = (R2*)aos;
    for (int32_t s = 0; s < nsteps; ++s)
        for (int64_t i = 0; i < n; ++i)
            for (int c = 0; c < 3; ++c) P[i].pos[c] = wrap(std::fma(dt, P[i].vel[c], P[i].pos[c]));
}

// ---- a8: ENERGY.  q = v0^2; q = fma(v1,v1,q); q = fma(v2,v2,q); [+ k d_c^2 terms]; e_i = 0.5 q ----------
//      kind 0 = kinetic, kind 1 = kinetic + harmonic.  For k = 1 the potential terms are fma(d,d,q) as in
//      SURVEY.md 8(c); the general form multiplies d*d by k first ("general: k*d^2").
static inline double energy_term(const double v[3], const double x[3], int kind, double k, double ctr) {
    double q = v[0] * v[0];
    q = std::fma(v[1], v[1], q);
    q = std::fma(v[2], v[2], q);
    if (kind == 1)
        for (int c = 0; c < 3; ++c) {
            double d = x[c] - ctr;
            q = std::fma(k * d, d, q);
        }
    return 0.5 * q;
}

double soax_oracle_r1_energy(const void* aos, int64_t n, int32_t kind, double k, double ctr) {
    const unsigned char* base = (const unsigned char*)aos;
    Neumaier acc;
    for (int64_t i = 0; i < n; ++i) {
        R1 p = load1(base, i);
        double v[3] = {(double)p.vel[0], (double)p.vel[1], (double)p.vel[2]};
        double x[3] = {p.pos[0], p.pos[1], p.pos[2]};  // copies: a pointer to the packed (4 mod 8) member would be misaligned
        acc.add(energy_term(v, x, kind, k, ctr));
    }
    return acc.value();
}

double soax_oracle_r2_energy(const void* aos, int64_t n, int32_t kind, double k, double ctr) {
    const R2* P = (const R2*)aos;
    Neumaier acc;
    for (int64_t i = 0; i < n; ++i) acc.add(energy_term(P[i].vel, P[i].pos, kind, k, ctr));
    return acc.value();
}

// ---- a6 / a7: AoS <-> SoA, a bit copy of each field of each record -----------------------
//      comp[0] = id, comp[1..3] = pos0..2, comp[4..6] = vel0..2: one contiguous array per component
//      (PAPER.md:155).
void soax_oracle_r1_aos_to_soa(const void* aos, int64_t n, int32_t* id, double* pos0, double* pos1, double* pos2,
                               float* vel0, float* vel1, float* vel2) {
    const unsigned char* base = (const unsigned char*)aos;
    double* pos[3] = {pos0, pos1, pos2};
    float* vel[3] = {vel0, vel1, vel2};
    for (int64_t i = 0; i < n; ++i) {
        R1 p = load1(base, i);
        id[i] = p.id;
        for (int c = 0; c < 3; ++c) { pos[c][i] = p.pos[c]; vel[c][i] = p.vel[c]; }
    }
}

void soax_oracle_r1_soa_to_aos(void* aos, int64_t n, const int32_t* id, const double* pos0, const double* pos1,
                               const double* pos2, const float* vel0, const float* vel1, const float* vel2) {
    unsigned char* base = (unsigned char*)aos;
    const double* pos[3] = {pos0, pos1, pos2};
    const float* vel[3] = {vel0, vel1, vel2};
    for (int64_t i = 0; i < n; ++i) {
        R1 p;
        p.id = id[i];
        for (int c = 0; c < 3; ++c) { p.pos[c] = pos[c][i]; p.vel[c] = vel[c][i]; }
        store1(base, i, p);
    }
}

// ---- a10..a13: cell index, per-cell counts, exclusive scan, stable rank -> gather permutation -----------
//      counts[cell]++ ; offsets = exclusive prefix sum ; perm = indices stably sorted by cell (Q12: gather
//      map, perm[j] = source index of the particle that ends in slot j) ; dest = its inverse.
//      Any of cell/counts/offsets/perm/dest may be null.  Returns 0, or -1 if a cell index is out of range.
int32_t soax_oracle_r1_bin(const void* aos, int64_t n, int32_t G, uint32_t* cell, uint32_t* counts,
                           uint32_t* offsets, uint32_t* perm, uint32_t* dest) {
    const unsigned char* base = (const unsigned char*)aos;
    const int64_t ncell = (int64_t)G * G * G;
    std::vector<uint32_t> cl((size_t)n), cnt((size_t)ncell, 0u), off((size_t)ncell, 0u);
    for (int64_t i = 0; i < n; ++i) {
        R1 p = load1(base, i);
        const double x[3] = {p.pos[0], p.pos[1], p.pos[2]};  // copies: no pointer into the packed record
        int64_t c = cell_of(x, G);
        if (c < 0 || c >= ncell) return -1;
        cl[(size_t)i] = (uint32_t)c;
        cnt[(size_t)c]++;
    }
    uint32_t run = 0;
    for (int64_t c = 0; c < ncell; ++c) { off[(size_t)c] = run; run += cnt[(size_t)c]; }
    if (cell) std::memcpy(cell, cl.data(), sizeof(uint32_t) * (size_t)n);
    if (counts) std::memcpy(counts, cnt.data(), sizeof(uint32_t) * (size_t)ncell);
    if (offsets) std::memcpy(offsets, off.data(), sizeof(uint32_t) * (size_t)ncell);
    if (perm || dest) {
        std::vector<uint32_t> next(off);                        // ascending i within a cell = stable
        for (int64_t i = 0; i < n; ++i) {
            uint32_t d = next[cl[(size_t)i]]++;
            if (dest) dest[i] = d;
            if (perm) perm[d] = (uint32_t)i;
        }
    }
    return 0;
}

// ---- a14: apply the permutation to every field: new[j] = old[perm[j]] -----------------------------------
void soax_oracle_r1_permute(const void* aos_old, void* aos_new, int64_t n, const uint32_t* perm) {
    const unsigned char* src = (const unsigned char*)aos_old;
    unsigned char* dst = (unsigned char*)aos_new;
    for (int64_t j = 0; j < n; ++j) store1(dst, j, load1(src, (int64_t)perm[j]));
}

// ---- NEXT-1: the paper's own benchmark: x += dt v on Particle<SIZE>, all float -------
//      Eq. 1 as printed has no wrap; the destination-type rule (Q2) makes it one float FMA per component.
void soax_oracle_b6_euler(void* aos, int64_t n, int32_t size_extra, float dt, int32_t nsteps) {
    float* base = (float*)aos;
    const int64_t stride = 6 + size_extra;                       // floats per record (24 B at SIZE=0)
    for (int32_t s = 0; s < nsteps; ++s)
        for (int64_t i = 0; i < n; ++i) {
            float* p = base + stride * i;
            for (int c = 0; c < 3; ++c) p[c] = std::fmaf(dt, p[3 + c], p[c]);
        }
}

// ---- NEXT-3: container operations on an array of structs of any record size ----------
// The paper's default removal: "the element to remove is overwritten by the last element", stated for
// ONE element.  For a set of flagged elements it is applied in the usual forward loop (Q20): walk i upwards;
// if element i is flagged, overwrite it (record AND flag) with the last element, shrink by one and look at slot i
// again -- the element that arrived may be flagged too.  `kill` is consumed (modified).  Returns the new length.
int64_t soax_oracle_remove_swap_last(void* aos, int64_t n, int64_t stride, uint8_t* kill) {
    unsigned char* a = (unsigned char*)aos;
    int64_t i = 0;
    while (i < n) {
        if (kill[i]) {
            if (i != n - 1) std::memcpy(a + i * stride, a + (n - 1) * stride, (size_t)stride);
            kill[i] = kill[n - 1];
            --n;
        } else {
            ++i;
        }
    }
    return n;
}
// Order-preserving removal: survivors keep their relative order.  Returns the new length.
int64_t soax_oracle_remove_stable(void* aos, int64_t n, int64_t stride, const uint8_t* kill) {
    unsigned char* a = (unsigned char*)aos;
    int64_t m = 0;
    for (int64_t i = 0; i < n; ++i)
        if (!kill[i]) {
            if (m != i) std::memmove(a + m * stride, a + i * stride, (size_t)stride);
            ++m;
        }
    return m;
}
// getElement(idx[k]) for k = 0..m-1: copies of whole records.
void soax_oracle_get_elements(const void* aos, int64_t stride, const uint32_t* idx, int64_t m, void* out) {
    const unsigned char* a = (const unsigned char*)aos;
    unsigned char* o = (unsigned char*)out;
    for (int64_t k = 0; k < m; ++k) std::memcpy(o + k * stride, a + (int64_t)idx[k] * stride, (size_t)stride);
}
// NEXT-4 (include/soax.h soax_gather_segments_aos): output row j is input row seg_src[i] + (j - seg_dst[i]), i the
// LAST segment with seg_dst[i] <= j.  The same row-by-row loop as oracle.gather_segments in Python (which stays, and pins
// this one in tests/test_container_oracle.py); written in C only so that 2^24 rows finish in seconds.
void soax_oracle_gather_segments(const void* aos, int64_t stride, const int64_t* seg_dst, const int64_t* seg_src, int64_t nseg,
                                 int64_t n, void* out) {
    const unsigned char* a = (const unsigned char*)aos;
    unsigned char* o = (unsigned char*)out;
    int64_t i = 0;
    for (int64_t j = 0; j < n; ++j) {
        while (i + 1 < nseg && seg_dst[i + 1] <= j) ++i;
        std::memcpy(o + j * stride, a + (seg_src[i] + (j - seg_dst[i])) * stride, (size_t)stride);
    }
}

// ---- NEXT-2: the one elementary operation numpy lacks, for oracle/expr.py: a correctly rounded fused multiply-add
//      over arrays (std::fma / std::fmaf are correctly rounded with or without hardware FMA).
void soax_oracle_fma_f64(const double* a, const double* b, const double* c, double* out, int64_t n) {
    for (int64_t i = 0; i < n; ++i) out[i] = std::fma(a[i], b[i], c[i]);
}
void soax_oracle_fma_f32(const float* a, const float* b, const float* c, float* out, int64_t n) {
    for (int64_t i = 0; i < n; ++i) out[i] = std::fmaf(a[i], b[i], c[i]);
}

}  // extern "C"
