/* wtide.h -- C ABI of libwtide (B200 / sm_100a).
 *
 * libwtide computes the time-dependent weighting-field correlation function H(x,t) of a 3D
 * diamond sensor with resistive graphitised column electrodes and evaluates the extended
 * Ramo-Shockley convolution of arxiv/paper_2605_13987 Eq. 1.1 for batches of drifting carriers.
 * Citations are PAPER.md line numbers (+ section); "Rn" are the readings listed in DESIGN.md.
 *
 * General rules
 *  - No exceptions, no global state except a thread-local error string (wt_last_error).
 *  - Return value 0 = WT_OK; negative = error and NO output is written.
 *  - The library never allocates device memory, never synchronises the stream, never touches the
 *    default stream.  All device buffers (H tables, trajectories, outputs, workspaces) are
 *    caller-owned device pointers (e.g. PyTorch tensors' data_ptr()); handles are library-owned
 *    HOST objects (wt_make_geometry does host work only and needs no GPU).
 *  - wt_solve_H and wt_convolve_currents ENQUEUE work on `cuda_stream` (a cudaStream_t passed as
 *    void*; must not be NULL / the legacy default stream) and return at once.  Sticky device
 *    errors surface at the caller's next synchronisation.
 *  - Units (R15): length um, time ns, potential V, charge e.  H is V/(um ns), velocity um/ns,
 *    currents e/ns.
 *  - H layout is part of the ABI:  H[ ((ix*ny + iy)*nz + iz)*nt + t ][3], fp32, time innermost,
 *    the three field components interleaved (BASELINE.json north_star (b)).
 */
#ifndef WTIDE_H
#define WTIDE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define WT_OK         0
#define WT_EINVAL    -1  /* null pointer, bad size, nt % 4 != 0, grid not 2^a 3^b, offsets not usable      */
#define WT_EGEOM     -2  /* no readout column, a column without node or pad node, pads of different
                            potential on one node                                                     */
#define WT_EUNSTABLE -3  /* `substeps` given and dt/substeps >= 2 eps / sigma_max  (R12)                 */
#define WT_ENOMEM    -4  /* workspace too small (size via wt_query / wt_conv_workspace_bytes)            */
#define WT_ECUDA     -5  /* a CUDA call or kernel launch failed                                          */

#define WT_BIAS    0     /* pad held at 0 V                         */
#define WT_READOUT 1     /* pad stepped to v_w at t = 0  (R2, R4)   */
#define WT_SEGMENT 2     /* conductive cylinder WITHOUT a contact pad: segments stacked on a pad column (same axis, other
                            z range, other resistivity) give a depth-dependent conductivity profile; where
                            columns overlap the first in the list wins (R13) */

typedef struct wt_geometry wt_geometry; /* opaque; created by wt_make_geometry, released by wt_free */

/* One graphitised column: a cylinder with its axis parallel to z (Fig. 7). */
typedef struct {
  double cx, cy;       /* axis position, um; any value, taken modulo the periodic box            */
  double radius;       /* um, > 0                                                                */
  double resistivity;  /* ohm*cm, > 0  (0.75 ohm cm for the test-beam sensor)      */
  double z0, z1;       /* depth extent, um, 0 <= z0 < z1 <= lz                                   */
  int    role;         /* WT_BIAS, WT_READOUT or WT_SEGMENT                                      */
  int    pad_at_z1;    /* 0: the contact pad is the column's first z-layer, 1: its last (R8); ignored for segments */
} wt_column;

/* "a text file describing the geometry of the conductive elements" as a C struct. */
typedef struct {
  double lx, ly, lz;   /* periodic box, um; lz = sensor thickness (R7)                           */
  int    nx, ny, nz;   /* grid; node i sits at (i*l)/n; each n = 2^a 3^b, even, 4 <= n <= 1024   */
  int    nt;           /* time samples of H, a multiple of 4                                      */
  double dt;           /* ns, output time step of H                                               */
  double eps_r;        /* relative permittivity (5.7 for diamond), uniform (R5)                   */
  double v_w;          /* normalisation potential, 1 V                              */
  int    substeps;     /* forward-Euler substeps per dt; 0 = auto = ceil(dt*sigma_max/eps) (R12)  */
  int    n_columns;
  const wt_column* columns; /* host array, borrowed for the duration of the call only            */
  int    mirror_z;     /* 0: the box is periodic in z (R7).  1: z = 0 and z = lz are mirror (Neumann) surfaces, by the method of
                          images: the handle describes the DOUBLED box lz' = 2 lz, nz' = 2 nz (node spacing
                          unchanged; nodes 0 and nz lie on the mirror planes) with the columns j < n_columns as given and
                          their images n_columns + j at z in [2 lz - z1, 2 lz - z0].  An image carries its own contact pad (on
                          the mirrored layer) unless the column's pad layer lies on a mirror plane (layer 0 or nz), where the
                          pad is its own image and the image column is a WT_SEGMENT.  Every query, table size and H layout is
                          that of the doubled box; the sensor is its first half, z in [0, lz] = layers 0 .. nz (layer nz
                          exists: interpolation up to z = lz needs no clamp).  Needs 2 nz <= 1024, 2 n_columns <= 127. */
} wt_geometry_desc;

/* Steps a0 (setup) of SURVEY.md section 8(a): voxelise the columns (node-centre test, minimum image
 * in x,y, first column wins on overlap; R13), collect the pad nodes, build the wavenumber tables,
 * the mixed-space fundamental-solution tables and the inverse of the bordered collocation matrix
 * (PAPER.md:64-65 voxelisation; :97 fundamental solution and boundary point charges; R8-R11).
 * Host work only, fp64.  *out is set only on success. */
int wt_make_geometry(const wt_geometry_desc* desc, wt_geometry** out);

/* Steps a1-a8: the pseudo-spectral forward-Euler solve of the quasi-static third-order PDE
 * div[eps grad d_t psi + sigma grad psi] = 0 (Fig. 3; R1-R20) for a
 * lock-step batch of `n_geoms` geometries on the SAME grid / nt (substeps may differ).
 *   geoms        host array of n_geoms handles
 *   H_dev        host array of n_geoms DEVICE pointers; table g receives H in the ABI layout,
 *                16-byte aligned, H_bytes_each >= WT_Q_H_BYTES
 *   workspace    device scratch, 256-byte aligned, >= sum over g of WT_Q_SOLVE_WORKSPACE_BYTES
 * H[n] = -grad_s(W[n] - W[n-1])/dt with W the response to the readout pads stepped to v_w (R2). */
int wt_solve_H(wt_geometry* const* geoms, int n_geoms, float* const* H_dev, size_t H_bytes_each,
               void* workspace_dev, size_t workspace_bytes, void* cuda_stream);

/* Steps a9-a12: Eq. 1.1 discretised on H's time grid (R21-R26):
 *   i_c[n] = -(q_c/v_w) sum_{m<=n, m<M_c} sum_a H~_a(x_c[m], n-m) v_{c,a}[m] dt,  n < nt,
 * H~ = trilinear blend of the 8 surrounding node rows with full fp32 weights (R23); indices and
 * fractions by wt_trajectory_nodes' arithmetic (R24).  Steps m >= nt are ignored (R26); a step
 * whose position or velocity is not finite contributes nothing.
 *   track_carrier_offsets_dev [n_tracks+1]   int64, carriers of track t = [off[t], off[t+1])
 *   carrier_step_offsets_dev  [n_carriers+1] int64, steps of carrier c = [off[c], off[c+1])
 *   pos_dev, vel_dev          [n_steps][3]   fp32, um and um/ns (v[m] is supplied by the caller, R22)
 *   charge_dev                [n_carriers]   fp32, e
 *   per_track 1: out_dev[n_tracks][nt] = sum over the track's carriers in carrier order (fixed
 *             order, run-to-run deterministic; R25);  0: out_dev[n_carriers][nt]
 *   workspace >= wt_conv_workspace_bytes(...), 256-byte aligned (may be NULL if that is 0)
 * Offsets must be non-decreasing with off[0] = 0 (not checked: the arrays live on the device). */
int wt_convolve_currents(const wt_geometry* geom, const float* H_dev,
                         int64_t n_tracks, const int64_t* track_carrier_offsets_dev,
                         int64_t n_carriers, const int64_t* carrier_step_offsets_dev,
                         const float* pos_dev, const float* vel_dev, const float* charge_dev,
                         int per_track, float* out_dev,
                         void* workspace_dev, size_t workspace_bytes, void* cuda_stream);

/* Eq. 1.1 summed per track (wt_convolve_currents with per_track = 1; Eq. 1.1, same arithmetic, same kernels, same
 * order of summation, bit-identical result) for callers that cannot allocate device memory: code in a tight serving loop,
 * harnesses that forbid cudaMalloc.  The per-carrier rows that the workspace form keeps in the caller's workspace live in a
 * device array built into the library: WT_NOALLOC_MAX_FLOATS fp32 = 4 MiB, held by every GPU that loads the library until
 * the process exits.  The call allocates nothing (no cudaMalloc, cudaFree or allocating library routine); the caller still
 * passes every input and the output, laid out as for wt_convolve_currents.
 *   limit      n_carriers * nt <= WT_NOALLOC_MAX_FLOATS (e.g. 4096 carriers at nt = 256, 1024 at nt = 1024); beyond it the call
 *              returns WT_ENOMEM, launches nothing and wt_last_error() names the limit: split the batch, or use the workspace form
 *   device     the device of cuda_stream must be current (its copy of the array is looked up on first use, once per device)
 *   sharing    every call on a device uses the same array.  Calls are safe back to back on one stream; two calls that may
 *              overlap on the GPU (different streams without an event between them, or host threads doing so) RACE on it
 *              and give wrong sums.  The array keeps the last call's rows; none of it has to start at zero, because each
 *              call writes every row it later reads.
 * Other errors as wt_convolve_currents. */
#define WT_NOALLOC_MAX_FLOATS (1 << 20)
int wt_convolve_tracks_noalloc(const wt_geometry* geom, const float* H_dev,
                               int64_t n_tracks, const int64_t* track_carrier_offsets_dev,
                               int64_t n_carriers, const int64_t* carrier_step_offsets_dev,
                               const float* pos_dev, const float* vel_dev, const float* charge_dev,
                               float* out_dev, void* cuda_stream);

/* Releases a handle returned by wt_make_geometry.  NULL is a no-op. */
void wt_free(void* handle);

/* ---- around the hot path ----------------------------- */

/* Static weighting field of a table, per volt of v_w:  Es[node][a] = dt * sum_n H[node][n][a]  (= -grad_s W[nt-1], the
 * telescoped response; R2).  es_dev: [nx*ny*nz][3] fp32 in the node order of the table. */
int wt_static_field(const wt_geometry* geom, const float* H_dev, float* es_dev, void* cuda_stream);

/* the electrostatic field of the sensor ("An iterative pseudo-spectral method ... is used
 * to solve the Laplace equation in the diamond sensor"; :95 V <-> rho by the 3-D FFT and a kernel that multiplies or divides by |k|^2;
 * Fig. 2 :107).  Reading R37: every node of column j (the voxel set of wt_make_geometry, all roles) is held at column_potentials[j],
 * there is no charge elsewhere, the box is periodic and neutral:  V(x) = c + sum_{s in S} q_s G(x - x_s), V = v_j on column j,
 * sum q = 0, G = fundamental solution of the spectral Laplacian with the Nyquist modes removed (R9, R11).  Solved by conjugate
 * gradients on the restricted operator in the neutral subspace, each step one V <-> rho round trip (forward 3-D DFT, times 1/|k|^2
 * or |k|^2, inverse 3-D DFT, restriction to the electrodes), the whole iteration in ONE cooperative kernel launch.
 *   column_potentials  HOST array [n_potentials], n_potentials = number of columns of the descriptor, volts
 *   precondition       0: plain CG;  1: preconditioned by the restricted Laplacian (the rho-from-V direction of Fig. 2)
 *   max_iter, tol      stop after max_iter steps or when |residual on the electrodes|_2 <= tol * |Pi v|_2
 *   V_dev              [nx][ny][nz] fp32 (node order of the H table), may be NULL
 *   E_dev              [nx*ny*nz][3] fp32 = -grad_s V in V/um, the layout wt_static_field writes (feeds wt_drift_* with
 *                      v_bias = 1), may be NULL (not both)
 *   info_dev           [4] fp64 on the device: iterations done (-1: the kernel gave up waiting for a lost CTA and the outputs
 *                      are not valid), |residual|_2/|Pi v|_2, the constant c, sum of the charges (library units)
 *   workspace          >= wt_static_workspace_bytes (41 bytes per node), 256-byte aligned
 * q is not unique (R37), V and E are.  Transforms in fp32, CG vectors and sums in fp64; run-to-run deterministic.
 * WT_EINVAL if an xy-plane of the grid does not fit in shared memory (nx*ny beyond about 24 000). */
int wt_static_workspace_bytes(const wt_geometry* geom, size_t* bytes);
int wt_solve_static(const wt_geometry* geom, const double* column_potentials, int n_potentials, int precondition, int max_iter,
                    double tol, float* V_dev, float* E_dev, double* info_dev, void* workspace_dev, size_t workspace_bytes,
                    void* cuda_stream);

/* Carrier transport in the solved field (PAPER.md:73 "computing the paths of the carriers", :101; BASELINE.json
 * configs[1] saturated-drift model), explicit Euler on H's time grid, fp32 in a fixed order (R35):
 *   E = v_bias * trilinear(Es, x)  (indices and fractions as wt_trajectory_nodes);  v = sign mu E / (1 + mu |E| / v_sat),
 *   mu = mu_e for sign < 0, mu_h for sign > 0;  x' = x + v dt;  recorded pos[m] = x, vel[m] = (x' - x)/dt  (R22).
 * A carrier records steps while 0 <= z <= lz and it is outside every column radius (minimum image in x, y), at most
 * max_steps.  Two calls, so that the caller can size the outputs (it reads offsets[n_carriers] in between):
 *   wt_drift_count          counts_dev[c] = number of steps of carrier c
 *   wt_offsets_from_counts  offsets_dev[0] = 0, offsets_dev[i+1] = counts[0] + ... + counts[i]   (CSR offsets of Eq. 1.1)
 *   wt_drift_fill           pos_dev / vel_dev [offsets[n_carriers]][3] in the layout wt_convolve_currents reads
 * start_dev [C][3] fp32 um, sign_dev [C] int8 (-1 electron, +1 hole); units um, ns, V (mu in um^2/(V ns), v_sat in um/ns).
 * workspace: >= wt_drift_workspace_bytes, 256-byte aligned. */
int wt_drift_workspace_bytes(const wt_geometry* geom, size_t* bytes);
int wt_drift_count(const wt_geometry* geom, const float* es_dev, double v_bias, double mu_e, double mu_h, double v_sat,
                   int64_t n_carriers, const float* start_dev, const int8_t* sign_dev, int max_steps, int64_t* counts_dev,
                   void* workspace_dev, size_t workspace_bytes, void* cuda_stream);
int wt_offsets_from_counts(int64_t n, const int64_t* counts_dev, int64_t* offsets_dev, void* cuda_stream);
int wt_drift_fill(const wt_geometry* geom, const float* es_dev, double v_bias, double mu_e, double mu_h, double v_sat,
                  int64_t n_carriers, const float* start_dev, const int8_t* sign_dev, int max_steps,
                  const int64_t* carrier_step_offsets_dev, float* pos_dev, float* vel_dev,
                  void* workspace_dev, size_t workspace_bytes, void* cuda_stream);

/* Electronics stage ("convolved with the transfer function of the front-end electronics, and noise is
 * added"):  out[r][n] = dt * sum_{j <= n, j < n_transfer} transfer[j] * currents[r][n - j]  (+ noise[r][n] if noise_dev),
 * t_cfd[r] = first crossing of cfd_fraction * (extremum of out[r] by absolute value) on the way to that extremum,
 * linearly interpolated, in units of dt; -1 for an all-zero row.  All arrays fp32 on the device; rows of nt samples. */
int wt_electronics(int64_t n_rows, int nt, const float* currents_dev, const float* transfer_dev, int n_transfer,
                   const float* noise_dev, double dt, double cfd_fraction, float* out_dev, float* t_cfd_dev, void* cuda_stream);

/* ---- helpers ------------------------------------------------------------------------------ */

/* Step a9 on its own (R24), for bit-exact index checks:  per step s
 *   inv = (float)((double)n/l);  u = x*inv (one fp32 multiply);  i0 = floorf(u);  f = u - i0;
 *   x,y: i0 mod n and (i0+1) mod n;  z: u clamped to [0, nz-1], i1 = min(i0+1, nz-1).
 * node0_dev[s][3] = (i0x, i0y, i0z), node1_dev[s][3] = (i1x, i1y, i1z), frac_dev[s][3] = f.
 * A non-finite position gives node0 = node1 = -1 and frac = 0. */
int wt_trajectory_nodes(const wt_geometry* geom, int64_t n_steps, const float* pos_dev,
                        int32_t* node0_dev, int32_t* node1_dev, float* frac_dev, void* cuda_stream);

int wt_conv_workspace_bytes(const wt_geometry* geom, int64_t n_tracks, int64_t n_carriers,
                            int per_track, size_t* bytes);

#define WT_Q_H_BYTES               1  /* nx*ny*nz*nt*3*4                                        */
#define WT_Q_SOLVE_WORKSPACE_BYTES 2  /* device scratch wt_solve_H needs for THIS geometry       */
#define WT_Q_SUBSTEPS              3  /* n_sub actually used                                     */
#define WT_Q_N_PADS                4  /* |B|, number of boundary point charges                   */
#define WT_Q_N_NODES               5  /* nx*ny*nz                                                */
#define WT_Q_N_CONDUCTING          6  /* nodes with sigma > 0                                    */
#define WT_Q_N_PAD_LAYERS          7  /* distinct z-layers holding pads                          */
#define WT_Q_NT                    8
#define WT_Q_N_COLUMNS             9  /* columns of the handle (2 n_columns of the descriptor with mirror_z)  */
#define WT_Q_NZ                   10  /* z layers of the handle (2 nz of the descriptor with mirror_z)        */
int wt_query(const wt_geometry* geom, int what, int64_t* value);

/* Host copies of setup results (for checks against an independent voxeliser):
 *   WT_A_COLUMN_ID     int8   [nx][ny][nz]   column index of the node, -1 = diamond
 *   WT_A_PAD_NODES     int32  [B][3]         (ix, iy, iz) in pad order (column, then ix, iy)
 *   WT_A_PAD_POTENTIAL double [B]
 *   WT_A_AINV          double [B][B]         upper-left block of the inverse bordered collocation matrix, pad order,
 *                                            in the library's units (eps = 1, unit voxel): the oracle's block / (eps * voxel volume)
 *   WT_A_GT, WT_A_GZT  float  [nx][nz][ny/2] mixed-space fundamental solution g~(kx, dz, ky) and its -d/dz
 * `bytes` must be exactly the array size. */
#define WT_A_COLUMN_ID     1
#define WT_A_PAD_NODES     2
#define WT_A_PAD_POTENTIAL 3
#define WT_A_AINV          4
#define WT_A_GT            5
#define WT_A_GZT           6
int wt_get_array(const wt_geometry* geom, int what, void* host_out, size_t bytes);

/* One line naming the execution wt_solve_H selects for this geometry on the current device (persistent kernel or
 * kernel chain, and which kernels), for logs and bench labels.  Needs no GPU for the chain; `out` is NUL-terminated. */
int wt_describe_plan(const wt_geometry* geom, char* out, size_t out_bytes);

/* Measured FP32 FMA rate of the current device in TFLOP/s (2 flops per FMA), for roofline reports: a short
 * register-resident FMA kernel on every SM, best of 5.  The ONLY call that waits for the device.
 * scratch_dev: device scratch of >= 1.25 MB. */
int wt_measure_fp32_fma(void* scratch_dev, size_t scratch_bytes, void* cuda_stream, double* tflops);

/* Number of CUDA kernels this process has launched through libwtide so far (bench.py reports the
 * difference over its timed region as "gpu_launches"). */
int64_t wt_launch_count(void);

/* Thread-local description of the last error on this thread ("" if none). */
const char* wt_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* WTIDE_H */
