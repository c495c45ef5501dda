/* psg_static.h -- ONE entry point of libpsg.so that allocates nothing.
 *
 * Why: some callers cannot call cudaMalloc -- code under CUDA graph capture, tight serving loops, harnesses that forbid it.
 * Every other call of include/psg.h works on a psg_ctx, and psg_create / psg_set_* allocate device memory.  This call
 * needs no context: the caller passes inputs and outputs, and the kernel's scratch memory (the per-block partial moments
 * that k_range_moments keeps in ctx memory) lives in a file-scope `static __device__` array inside the library.
 *
 * What it computes (Sec. 2.2, RadiusofGyration; PAPER.md:L188 for the barycenter): for every replica r the
 * weighted radius of gyration of ONE contiguous atom range [first_atom, first_atom + n_group_atoms),
 *     W = sum_i w_i,  c = sum_i w_i r_i / W,  Rg = sqrt(sum_i w_i |r_i|^2 / W - |c|^2)   (0 if the argument is <= 0),
 * the same numbers psg_cv_eval gives for a PSG_CV_RGYR CV (and PSG_CV_COM_COMPONENT CVs) over that range group, open
 * boundaries: the same thread -> atom map, the same binary64 moments, the same summation order.  No Jacobian, no bias.
 *
 * The limit: the scratch array holds PSG_STATIC_MAX_BLOCKS partial records of 5 binary64 moments (640 KiB; every GPU that
 * loads the library holds it until the process exits).  One record is one block of PSG_STATIC_TILE atoms of one replica:
 *     n_replicas * ceil(n_group_atoms / PSG_STATIC_TILE) <= PSG_STATIC_MAX_BLOCKS,
 * e.g. 16 replicas of 2,097,152 atoms or 1,024 replicas of 32,768.  Larger problems: PSG_ECAPACITY, nothing launched.
 *
 * Sharing: every call on a device uses the SAME array, and the array keeps the last call's contents.  A call overwrites
 * every record it later reads (nothing has to start at zero, and the counters of a ticket scheme are deliberately not used),
 * so calls in stream order are independent of what came before.  Two calls that OVERLAP on the GPU (different streams, or
 * two host threads on unordered streams) race on the array and give garbage: order them on one stream or with events.
 *
 * The call enqueues two kernels on `cuda_stream` and returns; it does not synchronise, and it calls no cudaMalloc, cudaFree
 * or allocating library routine (the first call on a device looks the array's device address up with
 * cudaGetSymbolAddress: no allocation either, but make that first call outside a graph capture). */
#ifndef PSG_STATIC_H
#define PSG_STATIC_H

#ifdef __cplusplus
extern "C" {
#endif

#define PSG_STATIC_TILE 2048        /* atoms per block = per partial record */
#define PSG_STATIC_MAX_BLOCKS 16384 /* partial records in the static scratch array (x 5 doubles = 640 KiB per GPU) */

/* device          : CUDA device ordinal, 0 <= device < 64; made current for the call, the caller's device is restored.
 * cuda_stream     : cudaStream_t of that device (NULL = the default stream).
 * d_pos           : DEVICE, positions, replica r's atom a at d_pos[(r * replica_stride_atoms + a) * pos_stride + {0,1,2}];
 *                   pos_stride 3 or 4 (4: 16-byte aligned float4 records, the 4th float is ignored).  Read only.
 * n_replicas      : R, 1 .. 65,535.   replica_stride_atoms >= first_atom + n_group_atoms.
 * first_atom, n_group_atoms : the range, n_group_atoms >= 1.
 * d_weight        : DEVICE, nullable: per-atom weights (masses) indexed by the atom index a, shared by all replicas;
 *                   NULL = 1.
 * d_xi            : DEVICE out, [R] float: Rg of each replica.
 * d_center        : DEVICE out, nullable, [R][4] double: c_x, c_y, c_z, W.
 * Ownership: all buffers stay the caller's; nothing is kept after the kernels ran.
 * Returns PSG_OK (0); PSG_EINVAL (-1) bad arguments; PSG_ECAPACITY (-4) beyond PSG_STATIC_MAX_BLOCKS; PSG_ECUDA (-3) a CUDA
 * error (no device, launch failure).  psg_static_last_error() gives the message of this thread's last failure. */
int psg_range_rgyr_static(int device, void* cuda_stream, const float* d_pos, int pos_stride, int n_replicas,
                          long long replica_stride_atoms, long long first_atom, long long n_group_atoms,
                          const float* d_weight, float* d_xi, double* d_center);

/* Message of the last psg_range_rgyr_static failure on this thread ("" if none).  Never NULL. */
const char* psg_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
