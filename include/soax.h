/* soax.h -- C ABI of the B200-native SoAx hot path (arXiv 1710.03462, "SoAx: A generic C++ Structure of
 * Arrays for handling particles in HPC codes").
 *
 * What the library is: per-particle streaming updates over heterogeneous particle records stored as a
 * Structure of Arrays (one contiguous device array per field COMPONENT, PAPER.md:95-116 Listings 2-3 and
 * PAPER.md:155 "three heap-allocated C++ arrays for x and v, respectively"), the AoS<->SoA transposition
 * (PAPER.md:118), a double-precision energy reduction and PIC-style cell binning with a permutation of every
 * field array, on one B200 (sm_100a).  Citations "PAPER.md:<line>" refer to the paper text;
 * "Qn" to the readings listed in DESIGN.md.
 *
 * Conventions (all calls):
 *   - plain C, no exceptions; every call returns an int status: SOAX_OK (0) or a negative soax_status;
 *   - pointers named dev_* are DEVICE pointers, host_* are HOST pointers, everything else is host memory;
 *   - the CALLER owns all device memory (PyTorch tensors in the harness); the library never calls cudaMalloc.
 *     soax_alloc only carves a caller-provided slab into aligned per-component arrays;
 *   - work is ENQUEUED on the caller's stream (`stream` = a cudaStream_t cast to void*, NULL = legacy default
 *     stream) and no call synchronises, except where stated; scalar results go to device pointers;
 *   - element counts are int64_t; permutations, counts and offsets are uint32_t device arrays (n < 2^32);
 *   - floating point is IEEE-754 binary64/binary32, round to nearest even, no fast-math; every fused
 *     multiply-add is explicit, so results are bit-reproducible.
 */
#ifndef SOAX_H
#define SOAX_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif
#if defined(__GNUC__)
#pragma GCC visibility push(default) /* the library is built with -fvisibility=hidden: only this header is exported */
#endif

typedef enum {
    SOAX_OK = 0,
    SOAX_ERR_INVALID_ARG = -1,    /* null pointer, negative size, misaligned buffer, n > capacity ...           */
    SOAX_ERR_UNKNOWN_LAYOUT = -2, /* the field list matches no compiled layout instantiation                    */
    SOAX_ERR_UNSUPPORTED = -3,    /* the operation needs a field (or a field type / dimension) the layout lacks:
                                     the run-time face of the paper's compile-time SFINAE check, PAPER.md:320   */
    SOAX_ERR_ALLOC = -4,          /* slab or scratch too small, or host allocation of a handle failed          */
    SOAX_ERR_CUDA = -5,           /* a CUDA runtime call failed; see soax_last_cuda_error()                     */
    SOAX_ERR_TOO_LARGE = -6       /* more particles than the fixed work area of soax_remove_stable_noalloc holds
                                     (SOAX_NOALLOC_MAX_N): use soax_remove with a scratch buffer of your own      */
} soax_status;

/* Element type of one field (id<int,1>, pos<double,3>, vel<double,3>, mass<float,1>). */
typedef enum { SOAX_I32 = 0, SOAX_I64 = 1, SOAX_U8 = 2, SOAX_F32 = 3, SOAX_F64 = 4 } soax_dtype;

/* One attribute of the particle record: the C face of SOAX_ATTRIBUTE(name, tag) plus its <type, dim> entry in
 * the std::tuple typedef (Listing 5).  dim = 1 (scalar) or 3 (vector), or any positive
 * count for the benchmark record's temp[SIZE] (Listing 4). */
typedef struct {
    const char* name;  /* "id", "pos", "vel", "acc", "mass", "charge", "flags", "temp" */
    int32_t dtype;     /* a soax_dtype */
    int32_t dim;
} soax_field;

typedef struct soax_layout soax_layout; /* opaque; owned by the registry, immutable, lives for the process  */
typedef struct soax_container soax_t;            /* opaque container: layout + n + capacity + component pointers    */

/* ---- layout registry (Listing 5; D7/D8 of the component inventory) ----------------------
 * Layouts are COMPILE-TIME typelists (csrc/layout.hpp) whose kernels are generated from C++ templates; this
 * call canonicalises a run-time field list (names, dtypes and dims, in declaration order) and returns the
 * matching instantiation.  Built in: R1 {int32 id; double pos[3]; float vel[3]}, R1R {double pos[3];
 * float vel[3]; int32 id} (the same record with naturally aligned AoS offsets: the Q1 sensitivity row), R2 {int64 id;
 * double pos[3]; double vel[3]; double acc[3]; float mass; float charge; uint8 flags} (BASELINE.json config
 * 4) and B6_S {float pos[3]; float vel[3]; float temp[S]} for S in {0, 8, 16, 32}.
 * Errors: INVALID_ARG (null, nfields <= 0, bad dtype/dim), UNKNOWN_LAYOUT. */
int soax_layout_define(const soax_field* fields, int32_t nfields, const soax_layout** out);

/* Run-time layouts.  The paper's container is generic over ANY attribute list; the compiled
 * registry above covers the records of the benchmark configs.  This call accepts any field list (names: C
 * identifiers, unique; sum of dims <= 48): if a compiled instantiation matches it is returned, otherwise a run-time
 * descriptor is created (an identical list returns the same handle).  A run-time layout supports the container
 * (soax_alloc, soax_field_ptr, soax_resize, soax_upload, soax_download, soax_copy, soax_layout_*) and user-written
 * fused programs (soax_expr_compile / soax_expr_run generate their kernel from the descriptor); the hand-written
 * kernel families (soax_step, transposes, energy, binning, removal, gather) answer UNSUPPORTED. */
int soax_layout_define_dynamic(const soax_field* fields, int32_t nfields, const soax_layout** out);

/* Number of fields / of component arrays (sum of dims) of a layout; negative status on error. */
int soax_layout_nfields(const soax_layout* layout);
int soax_layout_ncomp(const soax_layout* layout);
/* Describe component c (0 <= c < ncomp, declaration order, component-major): its field index, its index within
 * the field and its soax_dtype.  Any out pointer may be NULL. */
int soax_layout_comp(const soax_layout* layout, int32_t c, int32_t* field, int32_t* comp_in_field, int32_t* dtype);

/* Array-of-Structures image of the layout (D1): record stride in bytes and the byte offset of
 * every component.  packed != 0: declaration order, no padding (R1: stride 40, offsets 0 / 4,12,20 / 28,32,36 --
 * BASELINE.json config 3, reading Q1); packed == 0: natural C alignment.  comp_offsets has ncomp entries. */
int soax_layout_aos(const soax_layout* layout, int32_t packed, size_t* stride, size_t* comp_offsets);

/* Bytes of device memory soax_alloc needs for `capacity` particles (each component array starts on a 256-byte
 * boundary).  Returns 0 on error (null layout, capacity < 0). */
size_t soax_slab_bytes(const soax_layout* layout, int64_t capacity);

/* ---- container ("Soax<ArrayTypes> soax(42)", PAPER.md:110-116 allocate(n)) -----------------
 * Carve `dev_slab` (caller-owned device memory, 256-byte aligned, >= soax_slab_bytes(layout, capacity)) into
 * the per-component arrays and return a handle with n live particles.  The contents of the slab are not
 * touched.  The handle is host memory; release it with soax_free (which never frees the slab).
 * Errors: INVALID_ARG (null, n < 0, n > capacity, misaligned slab), ALLOC (slab too small). */
int soax_alloc(const soax_layout* layout, int64_t n, int64_t capacity, void* dev_slab, size_t slab_bytes,
               soax_t** out);
int soax_free(soax_t* s);
/* Live particle count; resize within capacity (PAPER.md:296 resize; no data movement).  Regrow is a CALLER-SIDE operation,
 * because the caller owns device memory: soax_alloc over a larger slab, soax_copy, soax_free of the old handle -- the Python
 * container does exactly that in Soax.reserve() / resize() / push_back_aos() with a growth factor of 1.5. */
int64_t soax_size(const soax_t* s);
int soax_resize(soax_t* s, int64_t n);
/* Device pointer of one component array: field f, component c -- the paper's posArr(c).
 * Errors: INVALID_ARG (bad field index), UNSUPPORTED (c outside the field's dimension). */
int soax_field_ptr(const soax_t* s, int32_t field, int32_t comp, void** dev_ptr);

/* Host <-> device transfer of whole component arrays (the end-to-end path: host buffers in, host buffers
 * out).  host_comps has ncomp entries, one host array of n elements per component (NULL entries are skipped);
 * copies are cudaMemcpyAsync on `stream` (truly asynchronous only from pinned host memory).  soax_upload sets
 * the live count to n (n <= capacity). */
int soax_upload(soax_t* s, const void* const* host_comps, int64_t n, void* stream);
int soax_download(const soax_t* s, void* const* host_comps, int64_t n, void* stream);

/* ---- a2..a4, a9: streaming integration steps (Eq. 1 "x += dt v") ------
 * box = [0,1)^3 with periodic wrap  wrap(x) = x - floor(x), a result of exactly 1.0 mapped to 0.0 (Q3).
 *   DRIFT                       pos_c = wrap(fma(dt, (double)vel_c, pos_c))                      (configs 1, 5)
 *   SYMPLECTIC_EULER_HARMONIC   vel_c = fma_V((V)dt, (V)(-(k*(pos_c - center))), vel_c), V = type of vel,
 *                               then DRIFT with the NEW vel (kick, then drift: Q2, Q4)           (configs 2, 3)
 *   RK2_MIDPOINT_HARMONIC_MASKED  only for particles with (flags & flag_mask) != 0:               (config 4)
 *                               w = k/(double)mass; a1 = -(w*(pos-center)); ph = wrap(fma(dt/2, vel, pos));
 *                               vh = fma(dt/2, a1, vel); a2 = -(w*(ph-center)); pos = wrap(fma(dt, vh, pos));
 *                               vel = fma(dt, a2, vel); acc = a2 (Q6, Q7, Q8); other particles: no change.
 *   EULER_NOWRAP                pos_c = fma_P((P)dt, vel_c, pos_c), P = type of pos: Eq. 1 exactly as printed,
 *                               no wrap (the paper's float benchmark)
 * Needs fields pos[3] (and vel[3]; RK2 also acc[3] double, mass float, flags uint8): otherwise UNSUPPORTED.
 * One full read-modify-write pass over memory per step and one kernel launch per step (Q14: no fusion in
 * time, as in the paper's "loop many times ... and average"). */
typedef enum {
    SOAX_STEP_DRIFT = 0,
    SOAX_STEP_SYMPLECTIC_EULER_HARMONIC = 1,
    SOAX_STEP_RK2_MIDPOINT_HARMONIC_MASKED = 2,
    SOAX_STEP_EULER_NOWRAP = 3
} soax_step_kind;

typedef struct {
    int32_t kind;      /* a soax_step_kind */
    uint8_t flag_mask; /* RK2: particle is active iff (flags & flag_mask) != 0; config 4 uses 1 */
    uint8_t pad_[3];
    double dt;
    double k;      /* spring constant (configs: 1) */
    double center; /* centre of the harmonic well (configs: 0.5) */
} soax_step_params;

/* nsteps passes over the n live particles of `s`, in place.  Errors: INVALID_ARG, UNSUPPORTED, CUDA.
 * With nsteps >= 2 on a capturable stream (any stream but the legacy default stream, not itself being captured)
 * the nsteps launches are captured once into a CUDA graph kept with the container and replayed by later identical
 * calls: the same kernels and passes, without a host round trip per step (what a launch-bound, L2-resident
 * particle set such as config 1 needs).  On the legacy default stream the launches are issued one by one. */
int soax_step(soax_t* s, const soax_step_params* params, int32_t nsteps, void* stream);

/* a5: the same arithmetic on an Array of Structures (packed image of `layout`, see soax_layout_aos), kept as
 * the in-library comparison baseline (thread per particle, strided access).  variant 0 = the
 * paper-faithful kernel (one thread per record, direct strided field access); variant 1 = best effort
 * (whole records staged through shared memory with coalesced 128-bit accesses).  dev_aos: n records,
 * 16-byte aligned.  Kinds DRIFT, SYMPLECTIC_EULER_HARMONIC and EULER_NOWRAP (the last also on the paper's float
 * record B6_S = Particle<SIZE>: the B200 re-run of Fig. 8). */
int soax_step_aos(const soax_layout* layout, void* dev_aos, int64_t n, const soax_step_params* params,
                  int32_t nsteps, int32_t variant, void* stream);

/* a6 / a7: bit copy of every field of every record between the packed AoS image and the component arrays
 * ("a function copying the array data for one index to the Particle member variables", bulk
 * form; PAPER.md:304 getElement).  dev_aos: n * stride bytes, 16-byte aligned.  aos_to_soa sets the live
 * count of dst to n (n <= capacity). */
int soax_aos_to_soa(soax_t* dst, const void* dev_aos, int64_t n, void* stream);
int soax_soa_to_aos(const soax_t* src, void* dev_aos, int64_t n, void* stream);

/* NEXT-4 ("MPI transfer of particle objects"): the merge of sorted runs of packed AoS records into the component
 * arrays of dst, written as a SEGMENTED GATHER: row j of dst (0 <= j < n) is record  dev_seg_src[i] + (j - dev_seg_dst[i])  of
 * dev_aos, where i is the LAST of the nseg segments with dev_seg_dst[i] <= j.  dev_seg_dst must start at 0 and be
 * non-decreasing (an empty segment repeats the next start); both tables are uint32 device arrays built by the caller from
 * counts (paper_1710_03462_b200/dist.py builds them from the all-gathered per-cell counts, so that `world` runs that are
 * each sorted by cell merge into one set sorted by (cell, run, position): one pass of 40 B read + 40 B written per particle
 * instead of a transpose plus a full sort).  The tables are trusted, on purpose (the call does not know how many records
 * dev_aos holds): a dev_seg_src entry that points past the source is the caller's error and reads out of bounds.  Only the
 * index arithmetic is made safe -- rows in front of dev_seg_dst[0] (a table that does not start at 0) are served from
 * segment 0 with offset 0, never from a negative index.  dst's live count becomes n. */
int soax_gather_segments_aos(soax_t* dst, const void* dev_aos, const uint32_t* dev_seg_dst, const uint32_t* dev_seg_src,
                             int64_t nseg, int64_t n, void* stream);

/* ---- a8: energy reduction in double -----------------------------------------------------------------------
 *   per particle  q = v0*v0; q = fma(v1,v1,q); q = fma(v2,v2,q)            (v_c = (double)vel_c)
 *   [+ HARMONIC:  d_c = pos_c - center; q = fma(k*d_c, d_c, q), c = 0,1,2]
 *   e_i = 0.5*q;  *dev_out = sum_i e_i  (double; fixed reduction tree: run-to-run deterministic)
 * dev_scratch: >= soax_energy_scratch_bytes() bytes, 8-byte aligned.  dev_out: one double on the device. */
typedef enum { SOAX_ENERGY_KINETIC = 0, SOAX_ENERGY_KINETIC_PLUS_HARMONIC = 1 } soax_energy_kind;
size_t soax_energy_scratch_bytes(void);
int soax_reduce_energy(const soax_t* s, int32_t kind, double k, double center, void* dev_scratch,
                       size_t scratch_bytes, double* dev_out, void* stream);

/* ---- a10..a14: PIC-style binning (BASELINE.json config 5) ------------------------------------
 *   cell_i    = (i0*G + i1)*G + i2,  i_c = (int32)(pos_c * G)  (x slowest; pos in [0,1): Q11, Q16)
 *   counts[c] = #{i : cell_i = c};  offsets = exclusive prefix sum of counts
 *   perm      = indices 0..n-1 stably sorted by cell (gather map: perm[j] = source index of the particle that
 *               ends in slot j; ties keep ascending index: Q12);  dst.f[j] = src.f[perm[j]] for EVERY component
 * The permutation is unique and the result is deterministic for any particle distribution.
 * grid_dim G: power of two, 1 <= G <= 64 (G^3 <= 2^18 cells).  src is read only; dst: same layout,
 * capacity >= n, must not alias src; its live count becomes n.  dev_counts, dev_offsets: G^3 uint32 each;
 * dev_perm: n uint32; any of the three may be NULL (a NULL dev_perm means no source index is carried through the passes;
 * NULL counts and offsets mean the sorted keys are not written).  dev_scratch: >= soax_scratch_bytes(layout, n, G) bytes,
 * 256-byte aligned.  Optional fusions (one call = config 5's whole pipeline): if drift_dt != 0 the particles are
 * DRIFTED by that dt on their way to dst -- dst = the drifted particles in cell order, binned by their drifted positions;
 * src is READ ONLY and keeps the pre-drift state (the drift is computed once for the keys and once more, with the same
 * fma, while the position arrays move: no pass over memory exists only to write positions back; Q22); if
 * dev_kinetic != NULL it receives sum_i 0.5*|vel_i|^2 as in soax_reduce_energy(KINETIC).
 * Errors: INVALID_ARG, UNSUPPORTED (no pos[3] double field, n >= 2^32), ALLOC (scratch too small), CUDA.
 * Positions outside [0,1) are a precondition violation: their cell index is clamped into the grid. */
size_t soax_scratch_bytes(const soax_layout* layout, int64_t n, int32_t grid_dim);
int soax_bin_permute(soax_t* src, soax_t* dst, int32_t grid_dim, double drift_dt, uint32_t* dev_counts,
                     uint32_t* dev_offsets, uint32_t* dev_perm, double* dev_kinetic, void* dev_scratch,
                     size_t scratch_bytes, void* stream);
/* The same operation IN PLACE: on return `s` holds its particles [drifted and] sorted by cell; `work` (same layout, capacity
 * >= n, must not alias s) is a work area whose contents are destroyed and whose live count does not change.  With src
 * read-only, two out-of-place passes need an intermediate copy of every record plus key and carried index in scratch
 * (48 B/particle for the 40-byte record); here the intermediate's 8-byte arrays live in `work`, the sorted set returns to
 * `s` in the second pass, and scratch holds only (key, index) and the paired 4-byte components: 24 B/particle for that record
 * (soax_scratch_bytes_inplace; 0 if unsupported).  Needs the default two-pass plan (16 <= G <= 64): UNSUPPORTED otherwise.
 * dev_perm[j] = the index particle j of the result had before the call.  Everything else as soax_bin_permute. */
size_t soax_scratch_bytes_inplace(const soax_layout* layout, int64_t n, int32_t grid_dim);
int soax_bin_permute_inplace(soax_t* s, soax_t* work, int32_t grid_dim, double drift_dt, uint32_t* dev_counts,
                             uint32_t* dev_offsets, uint32_t* dev_perm, double* dev_kinetic, void* dev_scratch,
                             size_t scratch_bytes, void* stream);


/* ---- NEXT-3: container operations on the device ---------------------------------
 * soax_remove deletes the particles whose byte in dev_kill (n bytes, one per live particle) is non-zero, from EVERY
 * component array:
 *   SOAX_REMOVE_SWAP_LAST  the paper's default, "the element to remove is overwritten by the last element"
 *                          (PAPER.md:175): in place (dst must be NULL), unordered.  For a set of flagged
 *                          particles the rule is applied in the usual forward loop (Q20): i walks up;
 *                          a flagged a[i] is overwritten by a[n-1], n shrinks, and slot i is examined again.
 *                          Equivalently: with m = n - #flagged, the k-th flagged slot below m (ascending)
 *                          receives the k-th surviving particle at or above m counted from the end; no other
 *                          row moves.
 *   SOAX_REMOVE_STABLE     order-preserving compaction into dst (same layout, no aliasing, capacity >= survivors;
 *                          s is left untouched).
 *   | SOAX_REMOVE_KEEP_FLAGGED  (ORed to either mode) the mask marks the particles that STAY: a particle is removed iff its
 *                          byte is ZERO.  One mask then serves both halves of a migration step (copy the leavers out:
 *                          STABLE | KEEP_FLAGGED; delete them in place: SWAP_LAST) without a second pass that writes its
 *                          complement.
 * The result is unique and deterministic for any mask.  The call is ASYNCHRONOUS like every other: the kernels read the
 * survivor count on the device, and the host learns it without a synchronisation in this call -- the counting kernel stores
 * it into a mapped pinned word owned by the target handle (s for SWAP_LAST, dst for STABLE) and the stream records an event;
 * the first later call that needs that handle's live count on the host (soax_size, or any call that launches over its
 * particles) waits for that one event, which completes after the two small counting kernels, not after the rows have moved.
 * While such a count is pending, use the target handle from ONE host thread only (the calls documented as read-only resolve
 * the count, i.e. write the handle); a call that gives the handle a new count (soax_resize, soax_upload, ...) first waits for
 * the pending one.  host_new_n: optional HOST pointer (NULL allowed) that also receives the survivor count by a
 * cudaMemcpyAsync on `stream`; give it PINNED memory -- with a pageable pointer that copy BLOCKS the host until both counting
 * kernels have run, which makes the call synchronous without any other sign; read it after synchronising the stream.
 * UNSUPPORTED while `stream` is being captured into a CUDA graph (the count event would never fire).
 * dev_scratch: >= soax_remove_scratch_bytes(n) bytes, 256-byte aligned; it must stay valid until the enqueued work is done.
 * STABLE into a destination whose capacity is below the survivor count: dst receives the survivors that fit and its live
 * count becomes its capacity; *host_new_n still reports the true count (a capacity >= n can never overflow).
 * Errors: INVALID_ARG, ALLOC (scratch too small), UNSUPPORTED (n >= 2^32), CUDA. */
typedef enum { SOAX_REMOVE_SWAP_LAST = 0, SOAX_REMOVE_STABLE = 1, SOAX_REMOVE_KEEP_FLAGGED = 4 } soax_remove_mode;
size_t soax_remove_scratch_bytes(int64_t n);
int soax_remove(soax_t* s, soax_t* dst, const uint8_t* dev_kill, int32_t mode, void* dev_scratch, size_t scratch_bytes,
                int64_t* host_new_n, void* stream);
/* Stable removal for callers that have NO device memory to offer as scratch and no means of getting any.
 * soax_remove leaves the scratch to the caller, which suits a host program that manages its own memory.  It does not suit
 * code that is merely handed the particle arrays: a diagnostics or load-balancing hook called from inside somebody else's
 * time step, where a cudaMalloc would stall every stream of the device and the memory budget belongs to the host code; a
 * simulation that has already given the whole of HBM to its particle slabs, so that an allocation would simply fail; a
 * plugin interface that passes device pointers through but exposes no allocator.  For those there is this ONE entry point,
 * which allocates nothing -- no device memory, no pinned memory, no event, on any call: its work area (per-tile and
 * per-segment counts of the mask, 68 bytes per 4096 rows) is an array compiled into the library, about 0.27 MB that every
 * GPU using the library keeps until the process ends.  That fixes the largest set it can serve:
 *     live(s) <= SOAX_NOALLOC_MAX_N = 2^24 particles; anything larger answers SOAX_ERR_TOO_LARGE and enqueues nothing.
 * What it computes is soax_remove(s, dst, dev_kill, SOAX_REMOVE_STABLE [| SOAX_REMOVE_KEEP_FLAGGED], ...) with the same
 * kernels: dst (same layout as s, no array shared with s) receives the surviving rows of s in their original order, s is
 * left as it was.  keep_flagged = 0: a non-zero mask byte removes the row; != 0: a non-zero byte keeps it.
 * Differences from soax_remove, all of them consequences of not allocating:
 *   - the survivor count is written to *dev_new_n, one int64 in DEVICE memory of the caller (required, 8-byte aligned);
 *     the handle-owned pinned word and event through which soax_remove reports it lazily would have to be created;
 *   - therefore dst's live count is NOT changed by this call.  Once the stream has passed the call (after the caller's own
 *     synchronisation or a copy of the word), set it with soax_resize(dst, min(count, capacity of dst)).  As with
 *     soax_remove, a destination smaller than the survivor count receives the survivors that fit, and the word still holds
 *     the true count;
 *   - the very first call on each device looks up the device address of the work area (one cudaGetSymbolAddress, with the
 *     caller's current device; nothing is allocated by it).  Make that first call outside any stream capture, and with the
 *     device that owns the containers current; later calls on that device only launch kernels;
 *   - ALL calls on one device share the one work area, which still holds whatever the previous call left in it.  Nothing
 *     in it needs clearing (each call overwrites every entry it reads later), but two calls whose kernels can run at the
 *     same time -- different streams without an ordering between them, or two host threads -- overwrite each other's
 *     counts and produce garbage.  Keep the calls of one device on one stream, or order them with events.
 * Errors: INVALID_ARG (null or aliasing handles, different layouts, null mask with n > 0, null or misaligned dev_new_n),
 * TOO_LARGE, UNSUPPORTED (layout without compiled kernels; device ordinal >= 64), CUDA.  n = 0 enqueues one 8-byte memset of
 * *dev_new_n and nothing else. */
#define SOAX_NOALLOC_MAX_N 16777216 /* 2^24 */
int soax_remove_stable_noalloc(const soax_t* s, soax_t* dst, const uint8_t* dev_kill, int32_t keep_flagged, int64_t* dev_new_n,
                               void* stream);
/* push_back of m particle objects (PAPER.md:304-307 `soax.push_back(particle)`): m packed AoS records (see
 * soax_layout_aos, 16-byte aligned) are appended behind the live particles; the live count grows by m.
 * ALLOC if n + m exceeds the capacity (the caller owns the memory: to regrow, soax_alloc a larger slab and
 * soax_copy into it -- the paper's resize). */
int soax_push_back_aos(soax_t* s, const void* dev_aos, int64_t m, void* stream);
/* Bulk getElement (PAPER.md:304 `soax.getElement(i)`): rows dev_idx[0..m) (uint32, each < n, repeats allowed) as m
 * packed AoS records in dev_aos (16-byte aligned).  An index >= n is not dereferenced: its record is all zero bytes. */
int soax_get_elements(const soax_t* s, const uint32_t* dev_idx, int64_t m, void* dev_aos, void* stream);
/* Copy the live particles of src into dst (same layout, capacity >= n); dst's live count becomes src's. */
int soax_copy(soax_t* dst, const soax_t* src, void* stream);

/* ---- NEXT-2: user-written fused element-wise programs ----------------
 * The paper lets the user write whole-array arithmetic, `soax.posArr(0) = soax.velArr(1) - soax.velArr(2)`
 * (PAPER.md:294), and fuses it with expression templates into one loop / one kernel without temporaries ("loop
 * fusion").  Here the user passes the program as TEXT; soax_expr_compile checks it
 * against the layout, generates ONE CUDA kernel for the whole program (every array it reads is loaded once with
 * 128/256-bit accesses, every array it assigns is stored once, 4 particles per thread like the built-in step
 * kernels) and compiles it for sm_100a with NVRTC; soax_expr_run launches it on the live particles.
 *   program := stmt { ';' stmt }       stmt := target ('=' | '+=' | '-=' | '*=' | '/=') expr
 *   target  := field | field[c]        a float or double field; a multi-component field without index expands the
 *                                      statement over its components c = 0, 1, ...; every other un-indexed
 *                                      multi-component field in it must have the same dimension and is read as its
 *                                      component c (scalar fields are read as they are)
 *   expr    := + - * / unary-  < <= > >= == !=  &  |  ( )  numbers  scalar names  field reads  and the calls
 *              fma(a,b,c) sqrt(x) abs(x) min(a,b) max(a,b) floor(x) wrap(x) float(x) double(x) select(cond,a,b) cell(G)
 * Precedence, lowest first: comparisons, '|', '&', + -, * /, unary -.  NOTE that '&' and '|' bind TIGHTER than comparisons
 * (Python's rule, not C's): `flags & 1 != 0` means `(flags & 1) != 0`, and conditions are joined WITH parentheses,
 * `(pos[0] < a) | (pos[0] >= b)`.  '&' takes two integers of the same type (or an integer literal) or two
 * conditions; '|' takes two conditions.  A binary operation on two integer LITERALS is evaluated in double (`1/2` is 0.5).
 * cell(G), G a literal power of two <= 64, is the int32 cell index of the particle on the G^3 grid, (i0*G + i1)*G + i2 with
 * i_c = (int32)(pos_c*G) clamped into [0, G-1] -- bit-equal to soax_bin_permute's (a10); it needs a field pos of 3 doubles.
 * Semantics: statements run in order for each particle and later statements see earlier assignments; typing is
 * C's: float op float is float, anything with a double is double, an assignment rounds to the target's type
 * (`a += b` is `a = (T)(a + b)`); named scalars and literals with a '.' or exponent are double, integer literals
 * take the type of the other operand; integer fields can only be compared, masked with '&', or converted with
 * float()/double(); wrap(x) is the periodic wrap into [0,1) of Q3.  Nothing is contracted: the only fused
 * multiply-adds are the fma() the user writes, division and sqrt are IEEE (-fmad=false -prec-div -prec-sqrt).
 * scalar_names: nscalars <= 16 names usable in the program; their values are passed to every run.
 * Errors: INVALID_ARG (syntax/type error, unknown name, wrong component index -- the run-time face of
 * PAPER.md:320; soax_expr_error() holds the message with the character position), UNSUPPORTED (NVRTC cannot be
 * loaded; set the environment variable SOAX_NVRTC to libnvrtc.so.12), CUDA.  Compilation needs no GPU; the code is
 * loaded onto the device at the first run.  soax_expr_run applies the program nsteps times (one launch and one
 * memory pass each; nsteps >= 2 on a capturable stream replays a captured graph, like soax_step): INVALID_ARG if
 * the container's layout is not the one the program was compiled for or nscalars differs. */
typedef struct soax_expr soax_expr; /* opaque compiled program; free with soax_expr_free */
int soax_expr_compile(const soax_layout* layout, const char* source, const char* const* scalar_names,
                      int32_t nscalars, soax_expr** out);
int soax_expr_run(soax_t* s, soax_expr* e, const double* scalars, int32_t nscalars, int32_t nsteps, void* stream);
int soax_expr_free(soax_expr* e);
/* User-written REDUCTIONS: `expression` is ONE expression of the same language (no assignment); its per-particle value,
 * converted to double, is summed over the live particles into *dev_out (device) with the fixed reduction tree of
 * soax_reduce_energy (a8): run-to-run deterministic, and an expression that restates the energy term operation by
 * operation reproduces soax_reduce_energy bit for bit.  dev_scratch: >= soax_energy_scratch_bytes() bytes, 8-byte
 * aligned.  A sum program cannot be passed to soax_expr_run, nor an assignment program to soax_expr_sum (INVALID_ARG). */
int soax_expr_compile_sum(const soax_layout* layout, const char* expression, const char* const* scalar_names,
                          int32_t nscalars, soax_expr** out);
int soax_expr_sum(const soax_t* s, soax_expr* e, const double* scalars, int32_t nscalars, void* dev_scratch,
                  size_t scratch_bytes, double* dev_out, void* stream);
/* User-written MASKS (what soax_remove consumes; PAPER.md:175 removal, 304-307): `condition` is ONE condition of the same
 * language -- a comparison, or comparisons joined by '&' and '|' -- e.g. "(flags & 1) != 0" or, for the particles that left
 * the cell range [lo, hi) of a slab decomposition, "(double(cell(64)) < lo) | (double(cell(64)) >= hi)".  soax_expr_mask
 * writes one byte per live particle into dev_mask (n bytes, 4-byte aligned): 1 where the condition holds, else 0, with the
 * access shape of the other generated kernels (4 particles per thread, one 32-bit store of 4 mask bytes).  Asynchronous.
 * A mask program cannot be passed to soax_expr_run / soax_expr_sum, nor the other kinds to soax_expr_mask (INVALID_ARG). */
int soax_expr_compile_mask(const soax_layout* layout, const char* condition, const char* const* scalar_names,
                           int32_t nscalars, soax_expr** out);
int soax_expr_mask(const soax_t* s, soax_expr* e, const double* scalars, int32_t nscalars, uint8_t* dev_mask, void* stream);
/* Message of the last failed soax_expr_compile on the calling thread ("" if none). */
const char* soax_expr_error(void);
/* The generated CUDA source (owned by the handle), for inspection. */
const char* soax_expr_cuda_source(const soax_expr* e);
/* Algorithmic bytes per particle the compiled kernel reads and writes (arrays read before being assigned /
 * arrays assigned): the roofline denominator of a user program. */
int soax_expr_traffic(const soax_expr* e, int32_t* bytes_read, int32_t* bytes_written);

/* ---- diagnostics ------------------------------------------------------------------------------------------ */
const char* soax_strerror(int status);
/* The cudaError_t (as int) of the last failed CUDA call made by this library on the calling thread, 0 if none. */
int soax_last_cuda_error(void);
/* Number of kernels this library has launched since load (or since the last soax_reset_launch_count). */
int64_t soax_launch_count(void);
void soax_reset_launch_count(void);
/* Launch-shape knobs for benchmarking sweeps ("step_ppt", "step_block", "step_persist", "xpose_*", "bin_bits", "bin_cluster",
 * "bin_csync", "bin_pace", ...); unknown keys return INVALID_ARG.  Not needed for normal use: defaults are the measured
 * best.  The knobs are process-global and NOT thread-safe: set them before the first call that launches work and do not
 * change them while another thread is inside the library (captured step graphs are keyed on the knobs and re-captured
 * when they change; soax_scratch_bytes follows "bin_bits", so query it after setting that knob). */
int soax_tune(const char* key, int64_t value);

#if defined(__GNUC__)
#pragma GCC visibility pop
#endif
#ifdef __cplusplus
}
#endif
#endif /* SOAX_H */
