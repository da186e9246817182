/*
 * gamma_b200.h -- C-ABI of libgamma_b200.so: the gamma-index hot path of arxiv/paper_1012_1900
 * (Gu, Jia, Jiang, "GPU-based fast gamma index calculation") for NVIDIA B200 (sm_100a).
 *
 * Citations are PAPER.md:<line> (+ section / equation / algorithm); "reading n" refers to the table of
 * readings in DESIGN.md.  Every entry point is plain C: raw pointers, sizes, a cudaStream_t passed as
 * void*.  Unless a parameter says HOST, pointers are DEVICE pointers owned by the caller (PyTorch in
 * the binding); the library never frees or modifies inputs.  The library owns grow-only device workspaces
 * (work lists, sort buffers, offset table): one for calls on the caller's stream, one per lane stream used by
 * back-to-back / batched calls (6), one for calls captured into a caller's CUDA graph, plus the staging buffers of
 * gamma_eval_host_batch; all released by gamma_release(), all counted by gamma_workspace_bytes().
 *
 * Conventions
 *   grids      dense fp32, x fastest: lin = ix + nx*(iy + ny*iz); reference and evaluation dose share
 *              one grid in every entry point except gamma_eval_general, where the evaluation
 *              dose has a grid of its own; an axis of size 1 is dropped (2D input; reading 12).
 *              N = nx*ny*nz must be < 2^31.
 *   result     gamma[N] fp32; voxels excluded by the low-dose cutoff (or with dD_v <= 0) hold NaN.
 *   async      all work is enqueued on `stream`; calls return without synchronising unless stated.
 *   errors     every int function returns GAMMA_OK (0) or a GAMMA_ERR_* code; on an argument error
 *              nothing is launched or written.  gamma_last_error_string() describes the last failure
 *              of the calling thread.  No exceptions, no abort.
 *   threads    calls are serialised by an internal mutex; consecutive calls on different streams are
 *              ordered by an event (they share the workspace).
 *   memory     workspace per voxel of the largest grid seen: 20 B up to 2^25 voxels (five u32 work lists), once for
 *              calls on the caller's stream and once per lane used by back-to-back / batched calls; larger grids first
 *              count their evaluated voxels M (one 4-byte read by the host, which SYNCHRONISES `stream` once inside
 *              the call) and take 20 B per EVALUATED voxel.
 *   no fallback: there is no CPU path; without a CUDA device every compute call returns GAMMA_ERR_CUDA.
 */
#ifndef GAMMA_B200_H
#define GAMMA_B200_H

#ifdef __cplusplus
extern "C" {
#endif

#define GAMMA_OK 0
#define GAMMA_ERR_INVALID_ARGUMENT 1
#define GAMMA_ERR_OUT_OF_MEMORY 2
#define GAMMA_ERR_CUDA 3

#define GAMMA_MODE_GLOBAL 0 /* dD = DD * D_norm                       (reading 8) */
#define GAMMA_MODE_LOCAL 1  /* dD_v = DD * D_r[v]                     (reading 9) */

/*
 * gamma_eval -- the per-reference-voxel gamma search (Eq. 1; Algorithm A1 steps 1-4,
 * PAPER.md:164-190; Algorithm A2 steps 2-7).
 *
 *   gamma[v] = min over the continuous evaluation surface of
 *              | (r_v/DTA, D_r[v]/dD) - (r_e/DTA, D_e(r_e)/dD) |
 * where the surface is the piecewise-linear interpolant of `eval` on the Kuhn split of every grid cell
 * (readings 5, 6) and the point-to-simplex distance is exact.  Cells are visited
 * in ascending order of their minimum spatial distance L and the search of a voxel stops when
 * L >= current gamma (readings 3, 4); there is no radius cap (reading 18).
 *
 *   ref, eval        DEVICE, N fp32 each
 *   dims             HOST, (nx, ny, nz), each >= 1, at least one > 1
 *   spacing_mm       HOST, (dx, dy, dz), each > 0
 *   DD               dose-difference criterion as a fraction (0.03 = 3 %), > 0
 *   DTA_mm           distance-to-agreement criterion in mm, > 0
 *   mode             GAMMA_MODE_GLOBAL | GAMMA_MODE_LOCAL
 *   low_dose_cutoff  in [0, 1): voxels with D_r < cutoff * D_norm are excluded (NaN); D_norm = max(ref)
 *                    (reading 10; the comparison is done in double so that it is decided identically
 *                    everywhere).  Excluded voxels still serve as evaluation points of their neighbours.
 *   out_gamma        DEVICE, N fp32, written entirely
 *   stream           cudaStream_t.  With the default options everything runs on `stream` (4 kernels).  Only with
 *                    opts.table_radius = 2 or a table_cap above 1024 the offset table is built on a library-owned
 *                    side stream that forks from and joins `stream` through events (legal under stream capture).
 *   (ordering)       A call behaves like one stream operation: its first kernel waits for the operation in front of it
 *                    before it reads ref / eval, and when its last kernel has completed, every earlier call has.
 *                    Consecutive calls can be OVERLAPPED instead: see gamma_opts::back_to_back.
 *   (CUDA graphs)    A call made while the CALLER is capturing `stream` becomes four kernel nodes and one memset node
 *                    of the caller's graph.  The graph holds addresses of a library workspace reserved for captured
 *                    calls: that workspace never moves afterwards (a later captured call that needs a larger one fails
 *                    with GAMMA_ERR_INVALID_ARGUMENT), gamma_release() frees it and thereby INVALIDATES every graph
 *                    that holds such nodes, and two graphs holding captured calls must not run concurrently (they
 *                    share that workspace; replays on one stream are ordered).  Direct calls never touch it.
 */
int gamma_eval(const float* ref, const float* eval, const int dims[3], const float spacing_mm[3], float DD,
               float DTA_mm, int mode, float low_dose_cutoff, float* out_gamma, void* stream);

/* Options of gamma_eval_ex / gamma_eval_host.  Zero-initialise, then set what differs. */
struct gamma_summary;
typedef struct gamma_opts {
    float norm_dose;      /* D_norm; <= 0: max(ref), found on the device (k_norm).  > 0 (e.g. the prescription dose,
                             PAPER.md:312): step a0 is not needed and, unless table_radius = 2, star_load >= 2 or
                             stats_* ask for k_norm's other results, the call is three kernels instead of four  */
    int presort;          /* pre-sort of the search work list (A2 step 3).  0: default (= 4);
                             1: one-pass MSD radix sort on the 8-bit key digit (32 steps per octave of the key);
                             2: no sort (Table 2's "without sorting"); 3: full LSD radix sort of the
                             `sort_key_bits` most significant key bits; 4: depth classes -- a 1-bit radix
                             sort done while the list is written: items whose key exceeds the first non-zero
                             table distance go to a list of their own and are searched first, a warp each
                             (adaptive lanes only; with lanes_per_voxel != 0 it means 1)                   */
    int star_phase;       /* 0: default (= 1); 1: interior voxels first try the 75 faces touching the voxel
                             and finish there when gamma_star <= distance to the rest of the surface;
                             2: off -- every voxel goes through the table search with key |DD|/dD, as in
                             Algorithm A2                                               */
    int lanes_per_voxel;  /* lanes that cooperate on one reference voxel in the table search.  0: default =
                             adaptive (a whole warp for the deep items at the head of the pre-sorted list,
                             8 lanes for the others; needs presort 1, 3 or 4, else 8); 1 = the paper's
                             thread-per-voxel mapping; 8; 32                               */
    int sort_key_bits;    /* presort = 3 only.  0: default (= 16); 8, 16, 24 or 32 most significant key bits   */
    long long table_cap;  /* 0: default (1024 with table_radius 1, 1<<20 with 2); max cells of the candidate box
                             of the sorted offset table (>= its entries); past the table the search
                             continues by exhaustive enumeration, so results never depend on it            */
    int profile_stages;   /* 1: record CUDA events between the stages of this call on `stream`, to be read
                             with gamma_get_stage_times (adds a few event records, no synchronisation)     */
    int graph;            /* 0: default (= 2); 1: the call goes out as ONE CUDA-graph launch: the library keeps an
                             instantiated graph of the call's kernels (captured once per kernel sequence, programmatic
                             edges included) and rewrites grid sizes and arguments of its kernel nodes for every call
                             (cudaGraphExecKernelNodeSetParams) -- a third of the host time of four stream launches; this
                             is also how back_to_back calls are launched.  Kernel sequences that cannot be rewritten in
                             place (side-stream table, full radix sort) replay a cached graph keyed by the exact
                             arguments, pointers included (96 are kept).  2: launch the kernels one by one.  Ignored
                             (= 2) while `stream` is being captured by the caller (the kernels then become nodes of the
                             caller's graph, with their own control block) and with profile_stages          */
    int table_radius;     /* 0: default (= 1); 1: the table is a data-independent PREFIX of the paper's table,
                             as far as table_cap allows, built beside a0 (nothing on the critical path);
                             2: the paper's radius max |DD| / dD (A1 steps 1-2), built once
                             a0's maxima exist                                                              */
    int interpolation;    /* 0: default (= 1); 1: the evaluation dose is the piecewise-linear surface on the Kuhn
                             simplices (the paper's method); 2: grid vertices only -- the classical discrete
                             gamma search (Low 1998), kept as an internal comparator: gamma_1 <= gamma_2 always
                             (same table walk and early exit; the star phase is off); 3: the same surface as 1,
                             but every cell of the table walk is evaluated as its six Kuhn tetrahedra with the
                             paper's routine: normal equations and recursion into the sub-simplices opposite
                             negative weights -- a slow variant kept to measure that trade
                             (3D grids; 2D / 1D grids use 1)                                              */
    int back_to_back;     /* 0: default.  1: the caller ASSERTS that nothing else has been enqueued on `stream` since the
                             library's previous call on it returned (no kernel, copy or event of the caller's, no other
                             library entry point).  Consecutive such calls are then run round-robin on 6 library-owned
                             streams, each with its own workspace and with grids of about half an SM's registers, so that
                             the kernels of different calls are resident together (one stream cannot do that: its
                             operations complete in order); each call goes out as one CUDA-graph launch.  `stream` stays the
                             ordering point: the first call of such a sequence starts after what is on `stream`, and `stream`
                             waits for every call, so whatever the caller enqueues afterwards sees all results.  Calls of
                             a sequence may COMPLETE out of order; a call that reads or writes a buffer an earlier call
                             of the sequence still writes (or writes one it reads) waits for that call -- the library
                             checks the ranges of ref / eval / out_gamma / stats_* -- so results are those of calls made
                             one after the other.  What the library cannot see is foreign work on `stream` between two
                             calls, hence the assertion.  Ignored (the call runs on `stream` itself) with
                             profile_stages, graph = 1, large tables, grids above 2^25 voxels and under stream capture */
    int star_load;        /* how the star phase gets its evaluation doses (BASELINE.json north_star (4)).
                             0: default (= 1); 1: compacted list -- k_classify writes the list of evaluated voxels,
                             k_star reads each voxel's 27 doses through L1 / L2, every evaluated voxel in flight at once
                             (4 kernels per call); 2: spatial tiles of 8 x 4 x 4 voxels plus a halo of one voxel staged
                             by the TMA into shared memory, two tiles in flight, classification, compaction and star
                             phase in ONE kernel (3 kernels per call; 3D grids with the default presort / star_phase;
                             needs nx % 4 == 0 and 16-byte aligned ref / eval, else it behaves as 3); 3: the same tile
                             kernel with the tiles filled by cooperative loads.  Same gamma, bit for bit; measured on
                             B200 the list is faster (profiles/r2_star_load.md), hence the default                  */
    int stats_nbins;      /* a6 fused into the call (all four stats_* fields; stats_hist = NULL: off).  The gamma
                             kernels accumulate, where they write gamma, what gamma_stats computes from the finished map:
                             same definition, same results (counts and histogram exact, sums in double), no second pass
                             over gamma[N].  1 <= stats_nbins <= 1024                                              */
    unsigned long long* stats_hist;        /* DEVICE, stats_nbins u64, overwritten                                  */
    struct gamma_summary* stats_summary;   /* DEVICE, one gamma_summary, overwritten                                */
    float stats_hist_max;                  /* > 0: bin b counts floor(gamma / stats_hist_max * stats_nbins) == b    */
} gamma_opts;

/* Several independent cases in one call (every reference voxel and every case is independent,
 * PAPER.md:141).  One case is tens of microseconds of dependent kernels that cannot fill 148 SMs; the batch spreads
 * the cases over 6 library-owned streams, each with its own workspace, so that their kernels overlap on the device
 * (the same mechanism as gamma_opts::back_to_back, for which the batch is shorthand).
 * Results are those of n_cases gamma_eval_ex calls, bit for bit.
 *   ref, eval, out_gamma   HOST arrays of n_cases DEVICE pointers (fp32, layout as in gamma_eval); the outputs must
 *                          not alias each other or any input (cases whose buffers overlap are run one after the other)
 *   dims, spacing_mm       HOST, n_cases x 3 (case-major); the criteria and options are shared by all cases
 *   opts                   as gamma_eval_ex, except: profile_stages and back_to_back are ignored (the cases always run on
 *                          the lanes), and stats_* cannot be honoured (one pair of buffers, n cases) -- passing stats_hist
 *                          or stats_summary returns GAMMA_ERR_INVALID_ARGUMENT; run gamma_stats on each map instead
 *   stream                 the batch starts after the work already on `stream` and `stream` continues after the last
 *                          case; asynchronous.  Cannot be captured into a CUDA graph (INVALID_ARGUMENT).
 * Errors: as gamma_eval; every case is checked before anything is enqueued.  n_cases = 0 is a no-op. */
int gamma_eval_batch(int n_cases, const float* const* ref, const float* const* eval, const int* dims,
                     const float* spacing_mm, float DD, float DTA_mm, int mode, float low_dose_cutoff,
                     const gamma_opts* opts, float* const* out_gamma, void* stream);

/* gamma_eval with options (opts may be NULL = defaults).  Same contract as gamma_eval. */
int gamma_eval_ex(const float* ref, const float* eval, const int dims[3], const float spacing_mm[3], float DD,
                  float DTA_mm, int mode, float low_dose_cutoff, const gamma_opts* opts, float* out_gamma,
                  void* stream);

/*
 * gamma_eval_general -- gamma with the evaluation dose on ITS OWN grid, and the closest point of the evaluation surface
 * (SURVEY.md 8(f) item 3).  Eq. 1 does not need the two doses on one grid (the paper's data were,
 * PAPER.md:312), and the refinements it cites (Stock et al. 2005: the "gamma angle" that tells a
 * dose-difference failure from a distance failure) need the point where the minimum is attained.
 *   The centre of reference voxel (i, j, k) is ref_origin_mm + (i, j, k) * ref_spacing_mm, evaluation vertex (i, j, k)
 *   sits at eval_origin_mm + (i, j, k) * eval_spacing_mm; the surface is the Kuhn interpolant of `eval` on its grid
 *   (readings 5, 6); gamma[v] = min over that surface of the distance of Eq. 1, exact (no radius cap, reading 18);
 *   a reference point outside the evaluation grid is compared with the surface as it is (no extrapolation, reading 11).
 *   ref            DEVICE, Nr = product of ref_dims fp32; ref_dims each >= 1
 *   eval           DEVICE, product of eval_dims fp32; every eval_dims >= 2 (three active axes)
 *   *_dims, *_spacing_mm (> 0), *_origin_mm (finite)   HOST, 3 values each (x, y, z)
 *   DD, DTA_mm, mode, low_dose_cutoff   as gamma_eval (D_norm = max(ref) unless opts->norm_dose > 0)
 *   opts           NULL or gamma_opts of which norm_dose and table_cap are used.  presort, star_phase, lanes_per_voxel,
 *                  sort_key_bits, profile_stages, graph, table_radius, interpolation, back_to_back and star_load are
 *                  IGNORED (this path has one kernel sequence); stats_hist / stats_summary return
 *                  GAMMA_ERR_INVALID_ARGUMENT (run gamma_stats on out_gamma)
 *   out_gamma      DEVICE, Nr fp32, written entirely (NaN = excluded)
 *   out_closest    DEVICE, Nr x 4 fp32 or NULL: (x, y, z in mm, evaluation dose) of one point of the surface at distance
 *                  gamma[v] (the minimiser need not be unique); NaN for excluded voxels.  The gamma angle follows as
 *                  atan2(|r - r_v| / DTA, |D - D_r[v]| / dD).
 *   stream         everything runs on `stream` (4 kernels + one memset), in stream order; cannot be captured.
 * With identical geometry the result equals gamma_eval's (other kernels, same surface); this path has no star / ring
 * shortcut because the reference point is not an evaluation vertex: every evaluated voxel walks the offset table,
 * 8 lanes per voxel.
 */
int gamma_eval_general(const float* ref, const int ref_dims[3], const float ref_spacing_mm[3], const float ref_origin_mm[3],
                       const float* eval, const int eval_dims[3], const float eval_spacing_mm[3],
                       const float eval_origin_mm[3], float DD, float DTA_mm, int mode, float low_dose_cutoff,
                       const gamma_opts* opts, float* out_gamma, float* out_closest, void* stream);

/*
 * gamma_eval_host -- the same computation for HOST buffers (A2 steps 1 and 8):
 * copies ref and eval to the device, runs gamma_eval_ex, copies gamma back and SYNCHRONISES `stream`
 * before returning.  ref_host, eval_host, out_gamma_host: HOST, N fp32 each (pinned memory makes the
 * copies asynchronous with respect to other streams).
 */
int gamma_eval_host(const float* ref_host, const float* eval_host, const int dims[3], const float spacing_mm[3],
                    float DD, float DTA_mm, int mode, float low_dose_cutoff, const gamma_opts* opts,
                    float* out_gamma_host, void* stream);

/*
 * gamma_eval_host_batch -- n_cases independent cases from HOST buffers with the transfers of A2 steps 1 and 8
 * overlapped with the computation: while case i is computed, the doses of case i + 1 travel to the
 * device and the gamma map of case i - 1 travels back (three rotating sets of device staging buffers, one library
 * stream per direction, the kernels on a third).  Arguments as gamma_eval_batch with HOST pointers (pinned memory makes
 * the copies asynchronous; pageable memory works, more slowly).  Starts after what is on `stream`, SYNCHRONISES before
 * returning; cannot be captured.  Results are those of gamma_eval_host case by case, bit for bit.
 * opts: as gamma_eval_batch (profile_stages, graph, back_to_back ignored; stats_* -> GAMMA_ERR_INVALID_ARGUMENT).  On a CUDA
 * error in the middle of the batch the call still waits for every copy it has enqueued before it returns the error, so the
 * caller's host buffers are no longer in use when it returns.
 */
int gamma_eval_host_batch(int n_cases, const float* const* ref_host, const float* const* eval_host, const int* dims,
                          const float* spacing_mm, float DD, float DTA_mm, int mode, float low_dose_cutoff,
                          const gamma_opts* opts, float* const* out_gamma_host, void* stream);

/* Summary written by gamma_stats (layout fixed, 48 bytes). */
typedef struct gamma_summary {
    unsigned long long n_eval; /* voxels with a finite gamma                                  */
    unsigned long long n_pass; /* of those, gamma <= 1                                        */
    double sum_gamma;          /* sum of gamma over evaluated voxels                          */
    double sum_gamma3;         /* sum of gamma^3: the paper's work predictor */
    float max_gamma;           /* 0 when n_eval == 0                                          */
    unsigned int n_nan;        /* excluded voxels (low 32 bits)                               */
    unsigned long long pad_;
} gamma_summary;

/*
 * gamma_stats -- pass rate / gamma histogram reduction (BASELINE.json north_star (5); not in the paper).
 *   gamma     DEVICE, n fp32 (NaN = excluded); may be NULL when n == 0
 *   nbins     1..4096; bin b counts finite gamma with floor(gamma / hist_max * nbins) == b, the last bin
 *             also takes everything >= hist_max
 *   hist_dev  DEVICE, nbins u64, overwritten;  out_dev: DEVICE, one gamma_summary, overwritten
 */
int gamma_stats(const float* gamma, long long n, int nbins, float hist_max, unsigned long long* hist_dev,
                gamma_summary* out_dev, void* stream);

/*
 * gamma_sort_pairs -- the hand-written LSD radix sort of the voxel work list (subsystem (3); PAPER.md:221,
 * 245 used Thrust): stable ascending sort of (key, value) pairs on key bits [begin_bit, end_bit).
 *   keys, vals  DEVICE, n u32 each, sorted in place;  n < 2^31; begin_bit, end_bit multiples of 8,
 *   0 <= begin_bit < end_bit <= 32.  Non-negative fp32 keys sort correctly as their bit patterns.
 */
int gamma_sort_pairs(unsigned int* keys, unsigned int* vals, long long n, int begin_bit, int end_bit,
                     void* stream);

/*
 * gamma_sort_pairs_noalloc -- gamma_sort_pairs for callers that cannot allocate device memory: same kernels, same
 * result bit for bit, but the second pair of buffers, the tile histograms and the element counter sit in an array that
 * is part of the library image instead of coming from cudaMalloc.  The call (first one included) issues no cudaMalloc,
 * cudaFree or other allocating routine; it enqueues kernels and, for an odd number of 8-bit passes, two device-to-device
 * copies on `stream`.
 *   Who needs it: code that runs while any thread of the process captures a stream in the global capture mode (the
 *   runtime refuses cudaMalloc there and the refusal invalidates the capture); code in a loop with a latency budget
 *   (cudaMalloc / cudaFree stall the whole device); and processes in which one pool owns the device memory (the PyTorch
 *   caching allocator, a planning system's arena), where an allocation behind the pool's back fails or fragments it.
 *   keys, vals, begin_bit, end_bit, stream   as gamma_sort_pairs; the device `stream` belongs to must be current
 *   n          0 <= n <= GAMMA_SORT_NOALLOC_MAX_PAIRS; a larger n returns GAMMA_ERR_INVALID_ARGUMENT (nothing is
 *              launched; the error string names the limit) -- such sorts need gamma_sort_pairs
 * Cost: the array takes about 8.3 MB (8 B per pair of the limit + 260 KB) of EVERY GPU on which the library's code gets
 * loaded, from then until the process exits, whether or not this function is ever called; gamma_release() does not
 * return it and gamma_workspace_bytes() does not count it.
 * First call on a device: looks up the array's address on that device (cudaGetSymbolAddress, once per device, may load
 * the library's module).  Make that first call outside any stream capture.
 * Sharing: all calls on a device use the same array, and it keeps what the last call left in it.  No part of it needs to
 * be zero on entry (every word a pass reads was written earlier in the same call), so nothing is cleared.  Two calls
 * whose kernels could overlap on the GPU -- different streams without an event between them, two host threads on two
 * streams -- RACE on it and give garbage; calls on one stream are ordered and safe.  Unlike the other entry points this
 * one is not ordered against the rest of the library by events: it touches none of the library's workspaces.
 */
#define GAMMA_SORT_NOALLOC_MAX_PAIRS (1 << 20)
int gamma_sort_pairs_noalloc(unsigned int* keys, unsigned int* vals, long long n, int begin_bit, int end_bit,
                             void* stream);

/*
 * gamma_offset_table -- the sorted offset table {n, L_n} (Algorithm A1 steps 2-3; A2
 * steps 4-5) with the cell bound of reading 4.  (Inside gamma_eval the radius is the
 * paper's max|DD|/dD over the grid, A1 step 1.)  By the symmetry L(o) = L(-o-1) the
 * table lists the octant m >= 0 only: entry (m, L^2), L^2 = sum_a (m_a h_a)^2, h = spacing/DTA, for every
 * m with m_a <= dims_a - 1 and L < radius, sorted ascending by (L^2 as fp32, then m_x + bx*(m_y + by*m_z));
 * the search expands each entry into its 8 (4 in 2D) offsets o_a in {m_a, -m_a-1}.
 *   out_entries  DEVICE, max_entries * 4 int32: (bits of L^2 as fp32, m_x, m_y, m_z) per entry
 *   out_count    DEVICE, 3 int32: number of entries written; 1 if the table was truncated to max_entries'
 *                worth of box (radius reduced), else 0; bits of the fp32 radius^2 actually covered
 */
int gamma_offset_table(const int dims[3], const float spacing_mm[3], float DTA_mm, float radius,
                       long long max_entries, int* out_entries, int* out_count, void* stream);

/* Counters of the last gamma_eval* call (SYNCHRONISES the stream of that call).  HOST outputs. */
typedef struct gamma_counters {
    long long n_voxels;      /* N                                                              */
    long long n_evaluated;   /* M: voxels that passed the cutoff                               */
    long long n_table_search;/* voxels that went through the sorted-table search               */
    long long table_entries; /* octant entries of the offset table                             */
    long long vertex_visits; /* owner vertices whose 26 faces were evaluated in the table search */
    float max_key;           /* radius of the table = largest key of the search list           */
    float norm_dose;         /* D_norm used                                                    */
    int table_truncated;
    int n_ring_search;    /* of n_table_search: voxels finished by the ring search (depth classes), no table walk */
    int pipelined;        /* 1: the call ran on a library lane stream (gamma_opts::back_to_back honoured, or a batch) */
    int pad_;
    long long calls_pipelined; /* such calls so far in this process                                               */
} gamma_counters;
int gamma_get_counters(gamma_counters* out_host);

/* Device time of each stage of the last gamma_eval* call made with opts.profile_stages = 1 (CUDA events on
 * the call's stream).  SYNCHRONISES that stream.  HOST output; milliseconds. */
typedef struct gamma_stage_times {
    float prep_ms;   /* a0 + A1 step 1 + a1: max(ref), max|DD|, cutoff + compaction (k_norm, k_classify) */
    float star_ms;   /* a1 + first part of a4: keys and the star phase (k_star)                  */
    float table_ms;  /* a3: offset table when it is built on the side stream (CONCURRENT with the main
                        stream); ~0 by default, where the table is built inside k_star (star_ms)   */
    float sort_ms;   /* a2: presort of the search work list                                      */
    float search_ms; /* a4 + a5: table search (ring + deep classes) and write-back               */
    float total_ms;  /* first event to last event on `stream` = prep + star + sort + search      */
} gamma_stage_times;
int gamma_get_stage_times(gamma_stage_times* out_host);

/* Number of CUDA kernels this library has launched in this process so far (host counter; memsets and
 * copies are not counted). */
long long gamma_launch_count(void);

/*
 * Device timeline of the kernels (diagnostic; only in a library built with -DGAMMA_TRACE, otherwise both calls return
 * GAMMA_ERR_INVALID_ARGUMENT).  gamma_trace_reset clears the records and switches the stamps on (SYNCHRONISES the
 * device); gamma_trace_read (SYNCHRONISES) copies them out: out_host HOST, 256 calls x 4 kernels (k_norm, k_classify,
 * k_star, k_table_search) x 4 u64 = (first thread started, dependency wait passed, last block ended, 0), nanoseconds
 * of %globaltimer, record of call number c (as counted on the single-call workspace) at index c % 256; *next_call =
 * number of the next call.  The timeline in profiles/ is made with bench_suite.py --suite trace.
 */
int gamma_trace_reset(void);
int gamma_trace_read(unsigned long long* out_host, long long* next_call);
/* The same build also keeps one record per warp of the LAST k_table_search launch: out_host HOST, max_warps (<= 8192)
 * x 8 u64 = (warp started, dependency wait passed, first work unit finished, warp ended, work units taken, 0, 0, 0),
 * warp w = block * 4 + warp in block; SYNCHRONISES.  Shows how long a work unit takes while every warp of the grid is
 * busy and how long when few are left (profiles/r2_profile.md). */
int gamma_trace_read_warps(unsigned long long* out_host, int max_warps);

/* Device memory the library's workspaces hold right now, in bytes (host counter): all workspaces and the staging buffers
 * of gamma_eval_host_batch; not the built-in scratch array of gamma_sort_pairs_noalloc (part of the library image). */
long long gamma_workspace_bytes(void);

/*
 * gamma_fp32_probe -- measures the plain-ALU FP32 rate of the device with independent FFMA chains
 * (the "alu" roofline denominator of bench.py; DESIGN.md section "Roofline").  SYNCHRONISES.
 *   out_tflops HOST: 2 * FFMA thread-instructions / second / 1e12, best of `repeats` launches.
 */
int gamma_fp32_probe(int repeats, double* out_tflops, void* stream);

/* Frees the workspace.  Safe to call at any time; the next call re-allocates. */
void gamma_release(void);

/* sizeof(gamma_opts), sizeof(gamma_summary), sizeof(gamma_counters), sizeof(gamma_stage_times) as compiled
 * into the library, for bindings to check their struct layouts against.  out_host: HOST, 4 ints. */
void gamma_abi_sizes(int out_host[4]);

/* Description of the last error seen by the calling thread ("" if none). */
const char* gamma_last_error_string(void);

/* Library version string, e.g. "gamma_b200 0.1 sm_100a". */
const char* gamma_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GAMMA_B200_H */
