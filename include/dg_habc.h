/* dg_habc.h — C ABI of the B200 nodal-DG + HABC time stepper (arXiv 1610.05023).
 *
 * One explicit LSRK4(5) time step of the nodal discontinuous Galerkin semi-discretisation of the acoustic
 * pressure-velocity system (eq (1a-b)) on an affine tetrahedral mesh of a cuboid, with the
 * multidimensional Padé high-order absorbing boundary condition on all six faces: 2D auxiliary solvers on
 * the faces, 1D on the edges, 0D compatibility systems at the corners (Algorithm 1).
 *
 * Symbols follow BASELINE.json: N = polynomial degree (the paper's P), J = number of auxiliary fields per
 * face (the paper's N), M = 2J+1.  Np = (N+1)(N+2)(N+3)/6, Nfp = (N+1)(N+2)/2 (Table 1).
 *
 * Conventions
 *   - every pointer argument is a HOST pointer unless its name ends in _dev;
 *   - interface arrays are float64, element-major [K][Np], in the library's node order (dg_get_nodes) and the
 *     caller's element order; the device layout (node-major, field-interleaved, fp64 or fp32) is private;
 *   - the library copies what it is given: the caller keeps ownership of every buffer it passes, and
 *     outputs are written into caller-allocated buffers;
 *   - every call returns DG_OK (0) or a negative DG_E* code; dg_last_error() returns the message of the
 *     last failing call on this thread;
 *   - all device work is enqueued on the stream given in dg_options (the CUDA stream handle, e.g.
 *     torch.cuda.current_stream().cuda_stream); dg_step is asynchronous, the dg_get_* calls synchronise.
 */
#ifndef DG_HABC_H
#define DG_HABC_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DG_OK 0
#define DG_EINVAL (-1) /* bad argument: N outside 1..8, J outside 0..12, NULL pointer, non-cuboid boundary */
#define DG_EMESH (-2)  /* degenerate or non-conforming mesh */
#define DG_ECUDA (-3)  /* CUDA runtime error (no device, launch failure, ...) */
#define DG_ENOMEM (-4) /* workspace too small / allocation failed */

typedef struct dg_solver dg_solver; /* opaque, owned by the library; free with dg_destroy */

/* dg_options.kernel: which kernel runs the fused 3D volume + surface + update stage (eq (41)-(43)).
 * All of them compute the same stage; they differ in how the D_r/D_s/D_t and LIFT contractions are carried out. */
#define DG_KERNEL_AUTO 0   /* fp64: MMA for N = 1, 2, 4, WS at N = 3, 5, TPG for N >= 6; fp32: ELEM for N <= 2, TF32 for
                              N = 3..5, TPG for N >= 6 */
#define DG_KERNEL_SCALAR 1 /* scalar FMA, operators in shared memory (or L1/L2 for high N); fp64 and fp32, N = 1..8 */
#define DG_KERNEL_MMA 2    /* fp64 DMMA (mma.sync.m8n8k4.f64), operator rows register-resident; N = 1..5 */
#define DG_KERNEL_WS 3     /* DG_KERNEL_MMA with warp-specialised loader / operand / MMA roles; fp64, N = 1..5 */
#define DG_KERNEL_TF32 4   /* fp32 on the tensor cores as error-compensated 3xTF32 (fp32-accurate); N = 3..5 */
#define DG_KERNEL_TPG 5    /* tensor-pipe kernels for the degrees whose operators do not fit the register file:
                              fp64 DMMA / fp32 3xTF32; N = 6..8 */
#define DG_KERNEL_ELEM 6   /* fp32, one thread per element, operators in constant memory; N = 1, 2 */

/* Tetrahedral mesh of a cuboid.  Any vertex order inside a tetrahedron is accepted
 * (negatively oriented cells are re-oriented internally).  The six planes bounding the vertex cloud are the
 * domain faces; each carries the HABC unless dg_options.face_bc says otherwise. */
typedef struct {
    int32_t nverts;
    const double* xyz;   /* [nverts][3] */
    int32_t ntets;
    const int32_t* tets; /* [ntets][4] */
} dg_mesh;

typedef struct {
    int32_t precision;        /* 64 or 32: arithmetic and storage type of the device state */
    double cfl;               /* multiplies the time-step rule, eq (46) PAPER.md:L796 (reading R7); <=0 means 1.0 */
    double dt;                /* > 0 overrides eq (46) */
    void* stream;             /* cudaStream_t, or NULL for the default stream */
    int32_t device;           /* CUDA device ordinal */
    void* workspace_dev;      /* optional DEVICE buffer (e.g. torch-allocated) of workspace_bytes; NULL: cudaMalloc */
    uint64_t workspace_bytes; /* size of workspace_dev; see dg_workspace_bytes */
    int32_t use_graph;        /* 1: replay the 5-stage step as a CUDA graph; ignored (plain launches) when stream is NULL,
                                 because the legacy default stream cannot be captured */
    int32_t kernel;           /* 3D kernel (one of DG_KERNEL_*): 0 = the library's choice for (precision, N).  A kernel
                                 that does not cover (N, precision) gives DG_EINVAL */
    int32_t face_bc[6];       /* boundary condition of the six domain faces, index axis * 2 + (1 for the face at the upper
                                 end of the axis): 0 = HABC (the default), 1 = p = 0 (free surface),
                                 2 = rigid wall (n.u = 0).  Auxiliary fields exist only on HABC faces, on the edges
                                 between two of them and at the corners where three meet */
    int32_t time_kernels;     /* 1: every step also records a CUDA event before and after the 3D kernel of each of its five
                                 stages, on the solver's stream and inside the replayed graph (no host synchronisation, no
                                 change to the kernels); read them with dg_last_step_kernel_ms.  0 (default): no events */
} dg_options;

typedef struct {
    int32_t N, J, K, Np, Nfp;
    int32_t T;        /* K^tri: boundary triangles */
    int32_t E;        /* K^lin: boundary lines */
    int32_t C;        /* K^pnt: corners */
    int32_t precision;
    int32_t launches_per_step; /* kernels launched by one time step (5 LSRK stages) */
    double dt;
    uint64_t device_bytes;     /* device memory held by the solver */
    int32_t kernel;            /* the 3D kernel in use (DG_KERNEL_*, never DG_KERNEL_AUTO) */
    char kernel_name[44];      /* a short label "<kernel><N>", e.g. "k_vol3d_ws<5>": the kernel's template name and the degree.
                                  A profiler prints the full instantiation (k_vol3d_mmag<6,2,8>, k_vol3d<double,5,4,4,true>),
                                  of which this is a prefix up to the first template argument */
} dg_info;

/* Device bytes dg_create needs for this problem (lets the caller allocate the workspace, e.g. with torch). */
int dg_workspace_bytes(const dg_mesh* mesh, int N, int J, int precision, uint64_t* bytes);

/* Build the solver: mesh hierarchy, reference operators (Warp & Blend nodes, D_r/D_s/D_t, LIFT; PAPER.md:L489,
 * L529), geometric factors, Padé coefficients c_n (eq (6)), inverse edge / corner matrices (L475), and
 * upload.  c, rho: [ntets], constant per cell.  opt == NULL: fp64, cfl 1, default stream,
 * device 0, CUDA graph on.  All fields start at zero. */
int dg_create(const dg_mesh* mesh, int N, int J, const double* c, const double* rho, const dg_options* opt,
              dg_solver** out);

int dg_get_info(const dg_solver* s, dg_info* out);

/* Physical coordinates of the nodes, [K][Np] each. */
int dg_get_nodes(const dg_solver* s, double* x, double* y, double* z);

/* Set p,u,v,w ([K][Np] each) and zero every auxiliary field (reading R5); the cached
 * incoming characteristics are initialised by running the closure chain once on the device. */
int dg_set_initial(dg_solver* s, const double* p, const double* u, const double* v, const double* w);

/* Point source delta(x - xyz) * amplitude * S(t) in the pressure equation, S(t) = (t - t_s)
 * exp(-pi^2 f_peak^2 (t - t_s)^2) being the time integral of the Ricker wavelet, eq (44).  The delta is projected
 * onto the cell that contains xyz (the first one, in the caller's order, whose barycentric coordinates are all
 * >= -1e-12).  Time starts at 0 at dg_set_initial; stage n of a step evaluates S at t + c_n dt (LSRK, L531-540).
 * amplitude = 0 switches the source off.  xyz: [3], host. */
int dg_set_source(dg_solver* s, const double* xyz, double f_peak, double t_s, double amplitude);

/* Advance nsteps time steps of 5 LSRK stages each (eq (42)-(43), L531-540; kernel order L627). Asynchronous. */
int dg_step(dg_solver* s, int nsteps);

/* Read back the volume fields ([K][Np] each; any pointer may be NULL) and, optionally, the PHYSICAL auxiliary
 * fields:  face_aux [T][J][3][Nfp] = p_i00 (eq (29)) and the two tangential velocities (in-plane Cartesian
 * axes in increasing order);  edge_aux [E][J*J][2][N+1] = p_ij0 (eq (32)) and the tangential velocity, set
 * index i*J+j with i <-> the face of lower normal axis.  Synchronises the stream. */
int dg_get_fields(dg_solver* s, double* p, double* u, double* v, double* w, double* face_aux, double* edge_aux);

/* Where the auxiliary cells are: per triangle (parent tet, local face, normal axis, outward sign), [T] each;
 * face_xyz [T][Nfp][3] node coordinates.  Any pointer may be NULL. */
int dg_get_face_map(const dg_solver* s, int32_t* tet, int32_t* face, int32_t* axis, int32_t* sign, double* face_xyz);

/* Per line: tangent axis [E], the two normal axes [E][2] (lower first) with outward signs [E][2];
 * edge_xyz [E][N+1][3] node coordinates.  Any pointer may be NULL. */
int dg_get_edge_map(const dg_solver* s, int32_t* axis, int32_t* normal_axes, int32_t* signs, double* edge_xyz);

/* Reference operators as the library computes them (host only, no device needed): rst [Np][dim],
 * D [dim][Np][Np] row-major, LIFT [Np][Nfaces*Nfp], Fmask [Nfaces][Nfp].  Any pointer may be NULL.
 * Returns Np through *np_out. */
int dg_reference_element(int dim, int N, double* rst, double* D, double* LIFT, int32_t* Fmask, int32_t* np_out);

/* Host-side hierarchy sizes without touching the device: counts[0..3] = K, T, E, C.  face_bc: NULL (HABC on all
 * faces) or the six codes of dg_options.face_bc. */
int dg_mesh_counts(const dg_mesh* mesh, const int32_t* face_bc, int32_t* counts);

/* Seconds of device time spent in each kernel family during the last dg_profile_step call (one time step run
 * with CUDA events around every launch; for per-kernel reporting, never inside a timed benchmark region).
 * ms[0..5] = volume+surface+update 3D, 2D update, 1D update, face closure, edge closure, corner closure. */
int dg_profile_step(dg_solver* s, double* ms);

/* Device time of the 3D kernel in each of the five LSRK stages of the LAST step that dg_step enqueued, from the events
 * of dg_options.time_kernels = 1 (DG_EINVAL without it or before the first step).  Unlike dg_profile_step this measures
 * the kernels where they really run: inside the timed region of a benchmark, back to back with the other kernels, in
 * the CUDA graph.  Synchronises the stream.  ms: [5], host. */
int dg_last_step_kernel_ms(dg_solver* s, double* ms);

/* Switch dg_options.time_kernels on or off on an existing solver (so that a benchmark can time its headline steps
 * without the event nodes and read the per-stage kernel times from a few further steps with them).  Synchronises the
 * stream and drops the captured step; the next dg_step captures it again.  The state is untouched. */
int dg_set_time_kernels(dg_solver* s, int on);

/* Raw device pointers of the current state, in the library's own layout (optional, lets a caller read
 * traces or fields on the device without the fp64 host round trip of dg_get_fields).  The pointers stay owned by the
 * library, are valid until dg_destroy, and hold the state reached by the work already enqueued on the solver's stream
 * (the caller orders its own reads after that stream).  dg_step flips the ping-pong buffers: call again after it.
 * elem_bytes = 8 (fp64) or 4 (fp32).  Layouts: q [K][Np][4] = (p,u,v,w) per node; face_aux [T][J][3][Nfp] holds the
 * ODE state p*_i and the two tangential velocities, and face_S [T][Nfp] the closure sum S = r^- + r^+ with
 * p_i00 = p*_i + S (eq (29)); edge_aux [E][J*J][2][N+1] holds p*_ij and the tangential velocity. */
typedef struct {
    int32_t elem_bytes;
    int32_t reserved;
    const void* q;
    const void* face_aux;
    const void* face_S;
    const void* edge_aux;
} dg_device_view;
int dg_get_device_ptrs(const dg_solver* s, dg_device_view* out);

/* dg_get_aux_fields_noalloc — the auxiliary-field read-back of dg_get_fields for callers that must not allocate.
 *
 * Who needs it.  dg_get_fields converts the face / edge auxiliary state to the physical fields p_i00 (eq (29),
 * PAPER.md:L384) and p_ij0 (eq (32)) in a device staging buffer before copying it to the host.  That staging
 * buffer is part of the solver's workspace, which somebody had to allocate: dg_create with cudaMalloc, or the caller
 * with its own allocator.  Some hosts can do neither at the moment they want the data: a process whose device memory
 * is handed out in full to another owner at start-up (a framework's caching pool, a fixed partition per tenant) and
 * has no allocator left to ask; a monitoring or checkpoint thread that runs while another thread of the process is in
 * a global-mode stream capture, during which cudaMalloc is an error; a time-critical loop that cannot take the
 * device-wide synchronisation cudaMalloc / cudaFree imply.  This call stages through a fixed array that lives inside
 * libdg_habc.so itself instead, so it asks nobody for memory.
 *
 * What it does.  Same result, bit for bit, as dg_get_fields(s, NULL, NULL, NULL, NULL, face_aux, edge_aux): face_aux
 * [T][J][3][Nfp], edge_aux [E][J*J][2][N+1], HOST buffers owned by the caller, either may be NULL.  The input is the
 * solver's current state (the work already enqueued on its stream is waited for); the call synchronises the stream
 * before it returns.  It calls no cudaMalloc, cudaFree, or any other routine that allocates device memory.
 *
 * The limit.  The staging array holds DG_NOALLOC_MAX_VALUES doubles (4 MiB).  It is a static __device__ array of the
 * library image, so every GPU on which the process uses the library carries these 4 MiB from the moment the library's
 * device code is loaded there until the process exits, whether this call is used or not.  A solver with
 * T*J*3*Nfp + E*J*J*2*(N+1) > DG_NOALLOC_MAX_VALUES gets DG_ENOMEM with a message that states both numbers, and
 * nothing is launched (configs[0] needs 3,648 values, configs[1] 153,600; use dg_get_fields above that).
 *
 * First call on a device.  The library looks up the array's device address once per device (cudaGetSymbolAddress,
 * with that device current) the first time the call is made for a solver on it.  Make that first call before any
 * stream capture begins in the process.
 *
 * Sharing.  All solvers of the process on one device stage through the same array, and it keeps whatever the last
 * call left in it.  Nothing needs clearing: each call overwrites exactly the values it then copies out and reads no
 * other.  Two calls in flight at once on one GPU would overwrite each other's staging data, so the library holds a
 * process-wide lock from the launch to the end of the copy-out; calls from several host threads therefore run one
 * after the other, and the caller must not defeat this from outside (e.g. by sharing one solver between threads). */
#define DG_NOALLOC_MAX_VALUES (1u << 19)
int dg_get_aux_fields_noalloc(dg_solver* s, double* face_aux, double* edge_aux);

const char* dg_last_error(void);
/* Waits for the solver's stream, then frees what the library owns (never the caller's workspace).  The stream given in
 * dg_options must still exist; the caller's current device is restored and no CUDA error state is left behind. */
void dg_destroy(dg_solver* s);

#ifdef __cplusplus
}
#endif
#endif /* DG_HABC_H */
