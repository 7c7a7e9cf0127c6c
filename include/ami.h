/* ami.h -- C ABI of the B200-native batched AMI evaluation path.
 *
 * What this library computes is defined by arXiv 2311.17189 (TorchAmi); citations are line
 * numbers of /root/reference/PAPER.md, "P<n>" are the readings listed in DESIGN.md.
 *
 *   ami_construct   host, one-time: labelled diagram R0 -> symbolic result of
 *                   the n nested Matsubara sums, Eqs. 1-5, stored as a flat term
 *                   table (unfactorised form of PAPER.md:100, Eq. 6) plus evaluation plans, with a
 *                   device-resident copy.
 *   ami_dispersion  kernel: internal momenta -> line energies, Eqs. 8-18, 2D
 *                   tight-binding dispersion.
 *   ami_evaluate    kernel: the table evaluated for a batch of energies x external frequencies x
 *                   inverse temperatures, complex128.
 *   ami_run         streamed driver: (generate or copy momenta) -> dispersion -> evaluate, chunked
 *                   and double-buffered over CUDA streams ("repeatedly call this
 *                   function for different energy batches", :291).
 *
 * Conventions
 *   - Every function returns int: 0 = AMI_OK, negative = error (see enum).  Nothing throws or
 *     aborts across this boundary.  ami_strerror() names a code, ami_last_cuda_error() gives the
 *     CUDA runtime's message for the last AMI_ECUDA on this thread.  (ami_tally_static also leaves
 *     the reason of its own refusals there.)
 *   - Pointers named d_* are DEVICE pointers owned by the caller (e.g. a torch tensor's
 *     data_ptr()); h_* and unprefixed array arguments are HOST pointers, read during the call
 *     only.  The library owns only ami_table objects.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Kernel
 *     entry points are asynchronous on it; host arrays they take are copied before returning.
 *   - complex128 = two doubles (re, im), interleaved.
 *   - The supplied energies are the NEGATIVE of the dispersion, e_i = -eps(k_i) (PAPER.md:84,
 *     :219); external frequencies come LAST in every alpha row.
 *   - There is no CPU fallback: a table built with device = -1 can be inspected and exported but
 *     every kernel entry point returns AMI_ECUDA for it.
 */
#ifndef AMI_B200_H
#define AMI_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  AMI_OK = 0,
  AMI_EINVAL = -1,             /* bad argument (null pointer, negative size, bad enum, ...) */
  AMI_EUNSUPPORTED_ALPHA = -2, /* |alpha_p| != 1 met at a summation (Eq. 4 is for +-1; P8) */
  AMI_ENOPOLE = -3,            /* a term with no line depending on nu_p (P9) */
  AMI_ECUDA = -4,              /* CUDA runtime error, or table has no device copy */
  AMI_ENOMEM = -5,             /* host or device allocation failed */
  AMI_EUNSUPPORTED = -6        /* valid request outside the built limits (see ami_limits) */
};

/* Built limits (compile-time constants of the kernels). */
enum {
  AMI_MAX_INT = 12,   /* internal sums m */
  AMI_MAX_EXT = 4,    /* external frequencies */
  AMI_MAX_EPS = 32,   /* energy symbols */
  AMI_MAX_DERIV = 6   /* highest Fermi/Bose derivative order */
};

typedef struct ami_table ami_table;

/* Which representation ami_evaluate executes. */
enum {
  AMI_PLAN_AUTO = 0,  /* the library's fastest plan for this table */
  AMI_PLAN_FLAT = 1,  /* the flat term table, term by term, table-driven (SURVEY 8(a) S3 as written) */
  AMI_PLAN_TREE = 3,  /* the Horner plan (terms grouped by denominator product, Fermi/Bose sums hash-consed
                         into a DAG) as a program interpreted by a table-driven kernel: node lists of uniform
                         multiply-add items, staged through shared memory in tiles with TMA; real energies.  What
                         AMI_PLAN_AUTO runs when the register plan is not available for the table */
  AMI_PLAN_REG = 2    /* specialised kernels: the table written out as straight-line code for this diagram
                         (terms grouped by denominator product, Fermi/Bose and denominator products in Horner
                         form), compiled with NVRTC on first use and cached on disk; real or complex energies.  Tables of
                         orders up to 6-7 become ONE kernel with every value in a register (register plan);
                         larger ones (order 7-8, 1e4-1e5 flat terms) are split: a leaf kernel, then the groups
                         of the Horner plan in parts of register-plan size evaluated by one launch (grid.y =
                         part), then a kernel that adds the parts (split plan).  ami_info.plan_kind says which */
};

/* Flag, OR-ed into the `plan` argument of ami_evaluate / ami_evaluate_momenta / ami_evaluate_momenta_lattice:
 * the caller states that this call is INDEPENDENT of the calls of this library issued right before it on the same
 * stream that carry the flag too (it reads nothing they write and writes nothing they read or write -- e.g. the
 * batches of a Monte-Carlo loop, each with its own momenta and result buffer, "repeatedly call this
 * function for different energy batches").  Such a run of calls may then execute beside one another: the
 * register-plan kernel of a flagged call does not wait for its predecessor before it starts, so the ramp of one batch
 * fills the SMs the tail of the previous one leaves idle (20-35 % more throughput for batches of 1e4-1e5 samples,
 * profiles/r02_batch_sweep.md).  Everything else keeps stream order: a flagged kernel COMPLETES only after its
 * predecessor has (it waits at its end), so an unflagged call, a copy, an event or any other work enqueued after a
 * run of flagged calls sees all of them finished, and a flagged call that follows work of another kind (a copy, a
 * kernel of the caller, an unflagged call) starts only when that has finished.  ALL calls of an uninterrupted run
 * of flagged calls are mutually unordered, not only neighbours: a loop that rotates over R buffer sets issues the
 * call that begins the reuse of a set WITHOUT the flag (every R-th call), which closes the run before it.
 * Ignored by the split plan and the table-driven plans (they stay ordered); refused by ami_run (AMI_EINVAL), which
 * orders its own chunks. */
#define AMI_PLAN_UNORDERED 0x100

enum { AMI_KIND_NONE = 0, AMI_KIND_REGISTER = 1, AMI_KIND_SPLIT = 2 };

typedef struct ami_info {
  int32_t n_int, n_ext, n_g, n_eps;
  int32_t n_fermi_leaves;   /* U_F: distinct (energy combination, sigma, derivative order) */
  int32_t n_den_leaves;     /* U_D: distinct denominators (oriented as produced, P10), excluding the unit leaf */
  int32_t max_deriv;        /* highest derivative order in the table */
  int32_t max_den_per_term; /* denominators per term (powers count as repeats) */
  int64_t n_terms;          /* T_flat after merging identical terms */
  int64_t n_terms_raw;      /* terms produced by the recursion before merging */
  int64_t n_multipoles;     /* pole groups with multiplicity > 1 met during construction */
  int64_t n_groups;         /* distinct denominator products R (Horner plan) */
  int64_t n_tree_nodes;     /* Fermi-trie nodes of the Horner plan, summed over groups */
  int64_t n_den_nodes;      /* denominator-trie nodes of the Horner plan */
  int64_t table_bytes;      /* bytes of the device-resident copy (all plans) */
  int64_t fp64_ops_flat;    /* FP64 instructions per (sample,frequency,beta) of the flat term loop */
  int64_t fp64_ops_tree;    /* same for the Horner plan with n_f = n_b = 1 (FT part + R part) */
  int64_t fp64_ops_tree_fermi; /* its frequency-independent part (FT sums and products under purely real denominators): once per (sample,beta) */
  int64_t fp64_ops_leaf_fermi; /* FP64 instructions per (sample,beta) of all Fermi/Bose leaves (common path) */
  int64_t fp64_ops_leaf_den;   /* FP64 instructions per (sample,beta,frequency) of the complex reciprocals */
  int64_t fp64_ops_dispersion; /* FP64 instructions per sample of ami_dispersion */
  int64_t fp64_ops_combos;     /* FP64 instructions done once per sample: distinct energy combinations of the leaves, reciprocals of purely real denominators */
  int64_t tree_plan_words;  /* program words of the tree plan (both programs), -1 = table outside its encoding */
  int64_t tree_plan_slots;  /* value slots (doubles) per sample the tree plan keeps */
  int32_t has_device_copy;
  int32_t reg_plan_status;  /* 0 = specialised kernels loaded, 1 = eligible, not compiled yet,
                               AMI_EUNSUPPORTED = table outside the specialised kernels' limits, other < 0 = error */
  int32_t plan_kind;        /* AMI_KIND_*: how AMI_PLAN_REG / AMI_PLAN_AUTO specialise this table */
  int32_t specialize_cached; /* 1 if the loaded kernels came from the on-disk cache */
  double specialize_ms;     /* host time ami_table_specialize (or the first evaluation) spent generating, compiling
                               (or fetching) and loading the kernels; 0 until then */
  /* register plan with several temperatures per launch: where it takes fewer instructions from two temperatures on,
     the R part is evaluated as Q(root) + sum_n Q(n) P_n, P_n the product of the complex reciprocals on the way to trie
     node n (once per frequency), Q(n) the per-temperature sums; otherwise in the Horner form of one temperature
     (then fp64_ops_mb_prefix = 0 and fp64_ops_mb_sum = the R part of fp64_ops_tree) */
  int64_t fp64_ops_mb_prefix; /* FP64 instructions per (sample,frequency) of the prefix products */
  int64_t fp64_ops_mb_sum;    /* FP64 instructions per (sample,beta,frequency) of the sum */
} ami_info;

/* ---- Diagram files (Fig. 2; "Feature: Feynman Graph Representation") ----------
 * A diagram file is plain text, one line of the diagram per row, four integers separated by blanks:
 *   source target is_fermion spin
 * source and target are vertex numbers 0..n-1, is_fermion is 1 for a fermionic line and 0 for a
 * bosonic (interaction) line, spin is a tag that is carried along.  A vertex that is
 * touched by exactly one row is the far end of an external leg (Fig. 2: vertices 0 and 1).  Text from
 * '#' to the end of a row is ignored. */
typedef struct ami_graph_edge {
  int32_t source, target, is_fermion, spin;
} ami_graph_edge;

/* read_graph: parses `text` (NUL-terminated).  With edges = NULL only counts the rows.
 * Errors: AMI_EINVAL for a row that is not four integers, a negative vertex, is_fermion outside
 * {0,1}, or more rows than `capacity`. */
int ami_graph_parse(const char* text, ami_graph_edge* edges, int32_t capacity, int32_t* n_edges);

/* label_graph + graph_to_R0: momentum/frequency-conserving labels for every line
 * and the R0 input of ami_construct.
 *   Legs: none (n_ext = 0) or one entering and one leaving leg of equal statistics (n_ext = 1; the
 *   external slot is the LAST column).  The part without the legs must be connected.
 *   A spanning tree is grown from the bosonic lines first, then the fermionic ones, in file order;
 *   the lines left over (chords, in file order) carry the independent labels e_0..e_{m-1}, every
 *   tree line follows from conservation at its vertices,
 *       sum_in alpha - sum_out alpha = 0   (legs included),
 *   by leaf stripping.  A bosonic chord would make an internal sum bosonic (Eq. 3 is the fermionic
 *   sum): AMI_EUNSUPPORTED.  R0 holds the fermionic lines that are not legs, in file order; bosonic
 *   lines carry no propagator here (contact interaction, reading P23).  Lines of equal alpha share
 *   one energy symbol whatever their spin tag (P7: the dispersion of this library has one band).
 * Outputs (any may be NULL; sizes are returned so that a first call can size the buffers):
 *   n_int, n_ext, n_g, n_eps
 *   alpha_all [n_edges][n_int + n_ext]  labels of every row of the file, legs and bosons included
 *   row_of_g  [n_g]                     which row of the file each R0 line is
 *   alpha     [n_g][n_int + n_ext], eps [n_g][n_eps], slot_is_fermionic [n_int + n_ext]: ami_construct's inputs
 *   cap_words: capacity, in int32 words, of EACH of alpha_all / alpha / eps (AMI_EINVAL if too small)
 * Errors: AMI_EINVAL (legs, connectivity, capacity), AMI_EUNSUPPORTED (bosonic chord, limits). */
int ami_graph_label(const ami_graph_edge* edges, int32_t n_edges, int32_t* n_int, int32_t* n_ext, int32_t* n_g,
                    int32_t* n_eps, int32_t* alpha_all, int32_t* row_of_g, int32_t* alpha, int32_t* eps,
                    uint8_t* slot_is_fermionic, int64_t cap_words);

/* ami_construct -- Eqs. 1-5, API of PAPER.md:246.
 *   n_int   number of Matsubara sums m (N_INT);  n_ext number of external frequencies (>= 0)
 *   n_g     number of Green's functions N in R0;  n_eps number of distinct energy symbols
 *   alpha   [n_g][n_int + n_ext] frequency coefficients, external LAST
 *   eps     [n_g][n_eps] energy coefficients; rows of R0 are unit vectors, lines with equal
 *           alpha must share a symbol so that a double pole is recognised
 *   slot_is_fermionic [n_int + n_ext]: statistics of each frequency slot (P5); internal slots
 *           must be fermionic (Eq. 3), else AMI_EINVAL
 *   sum_order [n_int] order of the sums, or NULL for 0..n_int-1
 *   prefactor the constant A of Eq. 6, usually 1
 *   device  CUDA device ordinal for the resident copy, or -1 for a host-only table
 *   out     receives the table; destroy with ami_table_destroy
 * Errors: AMI_EINVAL, AMI_EUNSUPPORTED_ALPHA, AMI_ENOPOLE, AMI_EUNSUPPORTED (limits), AMI_ENOMEM,
 * AMI_ECUDA. */
int ami_construct(int n_int, int n_ext, int n_g, int n_eps, const int32_t* alpha, const int32_t* eps,
                  const uint8_t* slot_is_fermionic, const int32_t* sum_order, double prefactor, int device,
                  ami_table** out);

int ami_table_info(const ami_table* tab, ami_info* info);

/* ami_search_sum_order -- which order of the Matsubara sums gives the smallest result
 * ("the order of integration"; the table size depends strongly on it, the value
 * does not).  Host only, no table is kept.  Orders are enumerated in lexicographic order starting
 * from 0..n_int-1; at most max_orders of them are constructed (<= 0: all n_int!).  Orders the
 * recursion rejects (AMI_EUNSUPPORTED_ALPHA, AMI_ENOPOLE, AMI_EUNSUPPORTED) are skipped.
 *   criterion 0: fewest flat terms T;  1: fewest FP64 operations per sample of the factorised
 *                (Horner) form, leaves included -- what the register plan executes
 *   best_order [n_int] out; best_cost, default_cost (cost of 0..n_int-1, -1 if rejected),
 *   n_tried (orders constructed successfully): optional outs.
 * Errors: AMI_EINVAL; when no enumerated order is accepted, the code of the last rejection. */
#define AMI_ORDER_FEWEST_TERMS 0
#define AMI_ORDER_FEWEST_OPS 1
int ami_search_sum_order(int n_int, int n_ext, int n_g, int n_eps, const int32_t* alpha, const int32_t* eps,
                         const uint8_t* slot_is_fermionic, int criterion, int64_t max_orders,
                         int32_t* best_order, int64_t* best_cost, int64_t* default_cost, int64_t* n_tried);

/* LaTeX of the flat term table (pretty_print_ft_terms): an `aligned` environment, one
 * term per row,   sign [coefficient] f_{s}^{(k)}(E) ... \frac{1}{(D)^{p}} ...   with
 *   f_{+}(E) = 1/(e^{beta E} + 1),  f_{-}(E) = 1/(-e^{beta E} + 1),  ^{(k)} the k-th derivative in E,
 *   E and D integer combinations of \epsilon_{i} (energy symbol i, the SUPPLIED energies, Eq. 2) and
 *   z_{j} (external frequency j, i nu or its continuation).  The regulator (P10) is not shown.
 * Call with buf = NULL to get the size (terminating NUL included) in *bytes. */
int ami_table_latex(const ami_table* tab, char* buf, size_t* bytes);

/* The same result in the factorised form the paper prints (PAPER.md:100-104, Eq. 6: FT * R; :115-132): terms grouped
 * by their denominator product R_g, the Fermi/Bose sums FT_g in Horner form with every sum that several groups share
 * named once (the library's Horner plan, i.e. what the specialised kernels execute):
 *   S_{n} ={}& [coef] f(..) [S_{child}] ...   one row per shared sum, children before parents
 *   I ={}& + S_{root(g)} \frac{1}{(D)^{p}} ...   one row per group
 * Far shorter than the flat table (order 6: 48 + ~230 rows of a few factors against 688 rows of 11).  Same notation
 * and buffer protocol as ami_table_latex. */
int ami_table_latex_factorized(const ami_table* tab, char* buf, size_t* bytes);

/* Serialises the flat table for inspection and tests.  Call with host_buf = NULL to get the size
 * in *bytes; then with a buffer of at least that size.  Layout (little endian, all int32 unless
 * noted): magic 'AMI1', n_int, n_ext, n_eps, U_F, U_D, T, m_f (Fermi factors per term = n_int),
 * n_d (denominator slots per term); then
 *   leafF_c   int32 [U_F][n_eps]   energy combination of each Fermi/Bose leaf
 *   leafF_sig int32 [U_F]          sigma = +1 / -1   (f_sigma(E) = 1/(sigma e^{beta E} + 1))
 *   leafF_k   int32 [U_F]          derivative order
 *   leafD_c   int32 [U_D][n_eps]   energy combination of each denominator
 *   leafD_a   int32 [U_D][n_ext]   external-frequency coefficients of each denominator
 *   fidx      int32 [T][m_f]       Fermi leaf of each factor
 *   didx      int32 [T][n_d]       denominator leaf of each factor, -1 = empty slot (factor 1)
 *   coef      float64 [T]          sign and rational prefactor of the term (without A)
 * The term value is A * coef * prod_a f^{(k)}_{sigma}(leafF_c . e) * prod_b 1/(leafD_a . z + leafD_c . e). */
int ami_table_export(const ami_table* tab, void* host_buf, size_t* bytes);

/* Serialises the tree plan's programs for inspection and tests (size query as above).  Layout: uint32
 * magic 'AMT1', n_words_beta, n_words_freq, n_consts, n_slots; code_beta[]; code_freq[]; pad to 8 bytes;
 * float64 consts[].  A program is a list of nodes: header word count << 16 | dst, then `count` item words
 * flag << 28 | a << 16 | b; DESIGN.md (6.3) says what a node computes. */
int ami_table_export_tree(const ami_table* tab, void* host_buf, size_t* bytes);

/* Frees the table, its device copy, its specialised kernels and the workspace of ami_run.  Waits for the work
 * outstanding on the table's device first (kernel entry points are asynchronous); NULL is accepted. */
void ami_table_destroy(ami_table* tab);

/* ami_dispersion -- Eqs. 8-18 for the 2D square lattice:
 *   K_i = sum_l alpha^i_l k_l + sum_x alpha^i_ext,x q_x,   e_i = 2 t (cos K_i,x + cos K_i,y) + mu
 * i.e. e_i = -eps(K_i) with eps(k) = -2t(cos kx + cos ky) - mu.
 *   d_k     momenta; component c (0 = x, 1 = y) of internal momentum l of sample s is at
 *           d_k[s * k_stride_sample + (2*l + c) * k_stride_comp].  The paper's layout (Eq. 8,
 *           row-major [N][2m]) is (2m, 1); SoA [2m][N] is (1, N).
 *   q       host [n_ext][2] external momenta;  t, mu: hopping and chemical potential
 *   d_e     out, float64 [n_eps][n] (SoA: sample index fastest) */
int ami_dispersion(const ami_table* tab, const double* d_k, int64_t k_stride_sample, int64_t k_stride_comp,
                   const double* q, double t, double mu, int64_t n, double* d_e, void* stream);

/* ami_dispersion_lattice -- the same map for momenta of dim = 1, 2 or 3 components (Eq. 14 is written for
 * any dimension d; Eq. 18's index range i*d .. i*d+d-1) and a choice of band (the paper leaves
 * eps_k to the user):
 *   AMI_BAND_TIGHT_BINDING  eps(K) = -2t sum_c cos K_c - mu   (hypercubic lattice; dim = 2 is ami_dispersion)
 *   AMI_BAND_FREE           eps(K) = t |K|^2 - mu             (free particles, t = 1/2m*)
 * and e_i = -eps(K_i) as above.
 *   d_k     component c of internal momentum l of sample s at d_k[s * k_stride_sample + (dim*l + c) * k_stride_comp]
 *   q       host [n_ext][dim];  d_e out, float64 [n_eps][n]
 * AMI_EINVAL for dim outside 1..3 or an unknown band.  ami_evaluate_momenta_lattice and ami_run (cfg.dim,
 * cfg.band) take the same choices in one fused kernel. */
enum { AMI_BAND_TIGHT_BINDING = 0, AMI_BAND_FREE = 1 };
int ami_dispersion_lattice(const ami_table* tab, const double* d_k, int64_t k_stride_sample, int64_t k_stride_comp,
                           const double* q, double t, double mu, int dim, int band, int64_t n, double* d_e,
                           void* stream);

/* ami_evaluate -- PAPER.md:106-113, :282-289.
 *   d_e     energies, [n_eps][n_e] float64, or complex128 if e_is_complex
 *   z_ext   host complex128 [n_f][n_ext]: external frequency values (i nu_ext on the Matsubara axis,
 *           omega + i Gamma after analytic continuation).  The paper's frequency_t rows
 *           also carry m internal placeholders; only the external columns are used (P13).
 *   beta    host [n_b] inverse temperatures (the paper's ami_vars holds one)
 *   e_reg   regulator eta, applied as in P10: added to the argument of every sigma = -1
 *           leaf and to every denominator whose frequency part is identically zero for that
 *           frequency; decided by table and frequency metadata only, never by sample values.
 *   plan    AMI_PLAN_*, optionally | AMI_PLAN_UNORDERED
 *   d_out   complex128 [n_b][n_f][n_e] (rows = frequencies, energy index fastest) */
int ami_evaluate(const ami_table* tab, const void* d_e, int e_is_complex, int64_t n_e, const double* z_ext,
                 int n_f, const double* beta, int n_b, double e_reg, int plan, void* d_out, void* stream);

/* Fused S1+S2+S3: ami_dispersion followed by ami_evaluate for the same samples in one call.  With the
 * register plan this is ONE kernel (the dispersion is inline and the energies never leave registers);
 * with the table-driven plans it is the two kernels back to back.
 *   d_k, strides, q, t, mu as for ami_dispersion;  z_ext, beta, e_reg, plan, d_out as for ami_evaluate
 *   d_e   float64 [n_eps][n] or NULL.  When given it receives the energies.  The table-driven plans
 *         need it as workspace and return AMI_EINVAL without it. */
int ami_evaluate_momenta(const ami_table* tab, const double* d_k, int64_t k_stride_sample, int64_t k_stride_comp,
                         const double* q, double t, double mu, int64_t n, const double* z_ext, int n_f,
                         const double* beta, int n_b, double e_reg, int plan, double* d_e, void* d_out, void* stream);

/* The fused call for momenta of dim = 1, 2 or 3 components and either band of ami_dispersion_lattice (Eq. 14 is
 * general in d; eps_k is the user's): d_k component c of internal momentum l of
 * sample s at d_k[s * k_stride_sample + (dim*l + c) * k_stride_comp], q host [n_ext][dim].  The specialised
 * kernels are generated per (dim, band), so this is ONE kernel like the 2-D call.  When d_e is NULL and a
 * table-driven plan runs, the energies live in a stream-ordered workspace of the library. */
int ami_evaluate_momenta_lattice(const ami_table* tab, const double* d_k, int64_t k_stride_sample,
                                 int64_t k_stride_comp, const double* q, double t, double mu, int dim, int band,
                                 int64_t n, const double* z_ext, int n_f, const double* beta, int n_b, double e_reg,
                                 int plan, double* d_e, void* d_out, void* stream);

/* Specialised kernels.  The compiled kernels are kept on disk under $AMI_JIT_CACHE, else
 * $XDG_CACHE_HOME/ami_b200, else $HOME/.cache/ami_b200, keyed by a hash of (generated source, NVRTC version,
 * architecture), so a second process on the same diagram loads them in milliseconds; AMI_JIT_CACHE=0 turns the
 * cache off.  ami_table_specialize compiles and loads the specialised kernels now
 * (otherwise this happens at the first evaluation with AMI_PLAN_AUTO or AMI_PLAN_REG); it returns
 * AMI_EUNSUPPORTED when the table is outside the plan's limits or NVRTC cannot be loaded, AMI_EINVAL when
 * compilation fails (ami_last_cuda_error() then holds the compiler log).  ami_table_kernel_source /
 * ami_table_kernel_cubin return the generated CUDA C++ text and its sm_100a cubin for inspection
 * (cuobjdump -sass); neither needs a GPU.  Call with buf = NULL to get the size for the source; for the
 * cubin pass a buffer and its capacity in *bytes (AMI_EINVAL if too small).  `log` (may be NULL) receives
 * the compiler log, including the ptxas resource usage lines. */
int ami_table_specialize(ami_table* tab);
int ami_table_kernel_source(const ami_table* tab, char* buf, size_t* bytes);
int ami_table_kernel_cubin(const ami_table* tab, void* buf, size_t* bytes, char* log, size_t log_cap);
/* A split plan is several translation units (the leaf and combine kernels first, then the parts, a few per unit,
 * compiled side by side): ami_table_kernel_units counts them, ami_table_kernel_source returns all of them one after
 * the other, ami_table_kernel_cubin_unit compiles unit `unit` (ami_table_kernel_cubin is unit 0). */
int ami_table_kernel_units(const ami_table* tab, int* n_units);
int ami_table_kernel_cubin_unit(const ami_table* tab, int unit, void* buf, size_t* bytes, char* log, size_t log_cap);
/* The kernels are generated per variant: lattice of the inline dispersion (dim, band as in ami_dispersion_lattice) and
 * real or complex energies (complex ones through ami_evaluate only: momenta give real energies).  The calls
 * above return the variant of the configurations (2, tight binding, real); these return any. */
int ami_table_kernel_source_variant(const ami_table* tab, int dim, int band, int complex_energies, char* buf,
                                    size_t* bytes);
int ami_table_kernel_cubin_variant(const ami_table* tab, int dim, int band, int complex_energies, int unit, void* buf,
                                   size_t* bytes, char* log, size_t log_cap);

/* Streamed driver.  Source of the momenta: if h_k / d_k are both NULL they are generated on the
 * device from `seed` with the counter-based generator of P22 (sample index = first_sample + s) --
 * with the register plan INSIDE the evaluation kernel, so the momenta never exist in memory; with
 * the table-driven plans by a generation kernel into a chunk buffer.  With the register plan and at
 * most 1024 result rows the tally is formed inside the evaluation kernel too (per-warp partial sums,
 * added in a fixed order), and per-sample results are written only if h_out / d_out is given;
 * else read from the given buffer, layout [n][2*n_int] (Eq. 8).  Results: per-sample values to
 * h_out / d_out (complex128 [n_b][n_f][n]) when given, and/or the running sum over samples to
 * h_sum (complex128 [n_b][n_f], Monte-Carlo tally of PAPER.md:291) when want_sum, with the sums of squares
 * to h_sumsq when that is given too (mean = sum/n, variance of the mean from sumsq/n - mean^2). */
typedef struct ami_run_cfg {
  int64_t n;             /* samples */
  int64_t chunk;         /* samples per chunk (0 = library default) */
  uint64_t seed;
  int64_t first_sample;
  const double* h_k;     /* host momenta or NULL */
  const double* d_k;     /* device momenta or NULL */
  const double* q;       /* host [n_ext][2] */
  double t, mu;
  const double* z_ext;   /* host complex128 [n_f][n_ext] */
  int32_t n_f;
  const double* beta;    /* host [n_b] */
  int32_t n_b;
  double e_reg;
  int32_t plan;
  int32_t want_sum;
  void* h_out;           /* host complex128 [n_b][n_f][n] or NULL */
  void* d_out;           /* device complex128 [n_b][n_f][n] or NULL */
  void* h_sum;           /* host complex128 [n_b][n_f] or NULL */
  void* stream;          /* caller's stream; internal copy/compute streams are ordered after it */
  void* h_sumsq;         /* host float64 [n_b][n_f][2] or NULL: sums of re^2 and im^2 over the samples (with
                            want_sum), for the Monte-Carlo error bar of the mean */
  int32_t dim;           /* components per momentum, 1..3 (0 = 2); momenta are [n][dim*n_int], q is [n_ext][dim] */
  int32_t band;          /* AMI_BAND_* of ami_dispersion_lattice (0 = tight binding) */
} ami_run_cfg;

typedef struct ami_run_stats {
  int64_t n_chunks;
  int64_t kernel_launches;  /* kernels of this library launched by the call */
  int64_t h2d_bytes, d2h_bytes;
  double gpu_ms;            /* CUDA-event time from first to last operation of the call */
} ami_run_stats;

int ami_run(const ami_table* tab, const ami_run_cfg* cfg, ami_run_stats* stats);

/* Fills d_k [n][2*n_int] with the momenta of samples first_sample .. first_sample+n-1 (P22); the _lattice
 * form for momenta of dim components, [n][dim*n_int] (counter of a component = sample * dim*n_int + index). */
int ami_generate_momenta(const ami_table* tab, uint64_t seed, int64_t first_sample, int64_t n, double* d_k,
                         void* stream);
int ami_generate_momenta_lattice(const ami_table* tab, uint64_t seed, int64_t first_sample, int64_t n, int dim,
                                 double* d_k, void* stream);

/* Register-only DFMA chains used by bench.py to measure the FP64 pipe of the device the bench runs on
 * (MEASURED_PEAKS.json has no FP64 figure).  distinct_sources = 2: x = fma(x, x, b), two different register
 * operands: the pipe's issue rate (0.995 of 148 SMs x 64 lanes x clock on B200), the roofline's peak.
 * distinct_sources = 3: x = fma(x, a, b), a and b shared by all chains: three different register operands of which two
 * repeat from one DFMA to the next (operand reuse): 0.92 of that.
 * distinct_sources = 4: x_i = fma(x_i, y_j, z_k) with y_j, z_k changing from one DFMA to the next: three different
 * register pairs and nothing to reuse -- 0.68 of the issue rate: the register file delivers one 64-bit operand per
 * lane and cycle, so such a DFMA occupies it for three cycles instead of two.
 * distinct_sources = 5: the same with one 32-bit integer instruction per two DFMAs (the proportion in the specialised
 * kernels): 0.54-0.60 -- integer instructions read the same register file.
 * distinct_sources = 6 / 7: x_i = fma(x_i, y_j, constant), two changing register operands and an immediate, without /
 * with the same integer work: 0.94 / 0.66.  (what these mean for the roofline fraction.)
 * Returns in *dfma_per_s the rate of double-precision FMA lane-operations per second. */
int ami_fp64_peak_probe(int device, int distinct_sources, double* dfma_per_s, double* elapsed_ms);

/* Allocation-free tally (the one entry point of this library that is safe where cudaMalloc is not: under CUDA
 * graph capture, in serving loops, in harnesses that forbid allocation).  Computes what ami_run's want_sum does
 * (Monte-Carlo tally of PAPER.md:291, error bar of :295) for results that are already on the device:
 *   d_tally[r] = (sum_i re v[r][i], sum_i im v[r][i], sum_i re^2, sum_i im^2),  r < n_rows,
 * v = d_vals, device complex128, row r starting at element r * row_stride (row_stride >= n; e.g. the
 * [n_b][n_f][n] result of ami_evaluate with n_rows = n_b * n_f, row_stride = n); d_tally: device double
 * [n_rows][4], every entry overwritten.  Deterministic: for given (n_rows, n) the order of every sum is fixed.
 * Asynchronous on `stream`; the call is one cudaMemsetAsync and one kernel, and calls no cudaMalloc, cudaFree or
 * any allocating routine.
 * Workspace: the per-block partial sums and the per-row arrival counters live in a file-scope device array of
 * AMI_TALLY_STATIC_BYTES (516 KiB) that every GPU on which the library is used holds until the process exits.
 * Limit: n_rows <= AMI_TALLY_STATIC_MAX_ROWS (1024), else AMI_EUNSUPPORTED with the reason in
 * ami_last_cuda_error(); n is not limited.
 * ALL calls on a device share that array: calls that may overlap on the GPU (different streams, parallel branches
 * of a graph, several host threads) race on it and give wrong sums -- order them on one stream or with events.
 * The counters are cleared by every call; nothing else of the previous call's contents is read.
 * The first call on a device looks the array's address up (cudaGetSymbolAddress, which may load the module):
 * call once with n_rows = 0 -- set-up only -- before starting a stream capture.
 * Errors: AMI_EINVAL (device outside 0..63, null pointer, negative size, row_stride < n), AMI_EUNSUPPORTED
 * (n_rows above the limit), AMI_ECUDA. */
#define AMI_TALLY_STATIC_MAX_ROWS 1024
#define AMI_TALLY_STATIC_BYTES (4096 + 16384 * 32)
int ami_tally_static(int device, const void* d_vals, int64_t n_rows, int64_t n, int64_t row_stride, double* d_tally,
                     void* stream);

/* Total number of kernels this library has launched in the calling process so far (all tables, all
 * streams); bench.py reports the difference over its timed region as "gpu_launches". */
int64_t ami_kernel_launches(void);

const char* ami_strerror(int code);
const char* ami_last_cuda_error(void);
int ami_version(void);

#ifdef __cplusplus
}
#endif
#endif /* AMI_B200_H */
