// td_f32.h - interface between tdlike.cu (the handle, the fp64 kernels) and tdlike_f32.cu, the translation unit that
// compiles the fused FFT-path kernels (td_fused4.cuh, td_cluster.cuh) a second time with real = float: the FP32
// evaluation mode of PAPER.md:322-324 (III.C.3: "carry out all the analysis with FP32 with appropriate normalization ...
// the necessary matrices and whitening operators should be precomputed in FP64").  Plain pointers only: the two units
// share no kernel types.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

#include "../../include/tdlike.h"

namespace td32api {

// size classes the fp32 kernels serve: M = 1024 .. 8192 on the fused / cluster kernels (segments of 513 .. 8192 samples), M >= 16384
// on the staged kernels (td_staged.cuh compiled with real = float: half the L2 traffic of a path that is bound by it)
inline bool supported(int log2M) { return log2M >= 10 && log2M <= 26; }
inline bool staged_class(int log2M) { return log2M >= 14; }

struct SegIn {
  long long off;      // offset of the segment inside d / a row of H (elements)
  int n;              // N_s
  int sid;            // index of the segment in the handle
  const void* Gp64;   // device double2 [2][padded(M)]: the fp64 generator spectrum in the padded Z layout (fused / cluster classes)
  const void* G64;    // device double2 [2][M]: the same spectrum in the plain layout (staged classes)
  double rho0;        // rho_s(0): samples are scaled by rho0^(-1/2) before rounding, the spectrum by rho0^(+1/2)
  const void* Gc64 = nullptr;   // device double2 [CS][padded(8192)]: per-CTA generator values of the group kernel (td_group16.cuh;
                                // classes 14..16, CS = M / 4096), or null
};

// device tables of one size class in fp32 (owned by the handle through this opaque record)
struct ClassTables {
  int log2M = 0, n_seg = 0;
  void* T = nullptr;        // float2 [2M] twiddles (rounded once from the fp64 table)
  void* segs = nullptr;     // td32::SegDev [n_seg]
  void* Gp_ptrs = nullptr;  // const float2* [n_seg]
  void** Gp = nullptr;      // host array [n_seg] of device float2 [2][padded(M)]
  void** zd = nullptr;      // host array [n_seg] of device float2 [M]
  void* host_segs = nullptr;  // staged classes: host copy of the td32::SegDev records
  void** Gc = nullptr;        // classes 14..16: host array [n_seg] of device float2 [CS][padded(8192)] (group kernel), entries may be null
};

// what a staged run borrows from the handle (td_staged_host.cuh: StagedCtx)
struct StagedBorrow {
  void* wsU = nullptr; size_t wsU_bytes = 0;
  void* wsZ = nullptr; size_t wsZ_bytes = 0;
  double* wsPartial = nullptr; size_t wsP_elems = 0;
  cudaStream_t aux_stream = nullptr;
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  int* launches = nullptr;
  unsigned* grp_bar = nullptr;   // arrival counters of the group kernel (td_group16.cuh)
  int group_cap = 0;             // groups the exchange buffers (wsU / wsZ) hold; 0: run the staged kernels
};

// builds the fp32 tables of a class from the fp64 ones (T64: device double2 [2M]); synchronous
td_status build_class(int log2M, int n_seg, const SegIn* segs, const void* T64, ClassTables* out);
void free_class(ClassTables* t);

struct Launch {
  const double* d;
  const double* H;
  long long ldh, B;
  double* out0;
  double* out1;
  int accumulate;
  int mode;  // td::MODE_LOGLIKE / MODE_INNER / MODE_STOREZ
  const StagedBorrow* staged = nullptr;   // staged classes only
  int syn = 0;      // 1: H holds ringdown parameter rows (ldh = 5 x segments of the handle), fused4 classes, MODE_LOGLIKE only
  double fs = 0.0;  // sampling rate (syn only)
};
// one launch of the class's kernel (dry: configure only - attribute, occupancy cache)
td_status launch(const ClassTables& t, const Launch& L, int num_sms, int device, cudaStream_t st, bool dry);

}  // namespace td32api
