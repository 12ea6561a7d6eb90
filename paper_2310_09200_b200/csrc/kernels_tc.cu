// tcgen05 (3xTF32) variant of the fused Standard Synthesizer — placeholder until the tensor-core
// kernel lands: the plan reports "no chunks", so creating work with BB_VARIANT_TF32X3 fails with
// BB_EUNSUPPORTED (loudly; never a silent fallback to the FP32 kernel).
#include "internal.h"

TcPlan bb_tc_plan(int, int, int) { return TcPlan{}; }
int bb_launch_prep_tc(const TcPlan&, const PrepArgs&, cudaStream_t) { return BB_EUNSUPPORTED; }
int bb_launch_synth_tc(const TcPlan&, const SynthArgs&, int, cudaStream_t, int* launches) { *launches = 0; return BB_EUNSUPPORTED; }
