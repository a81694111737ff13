// Instantiation unit of compact_inst.inc: confidence estimator 1, abstention on.
#define MOSAIC_INST_CONF 1
#define MOSAIC_INST_ABSTAIN 1
#define MOSAIC_INST_NAME dispatch_gate_c1a1
#include "compact_inst.inc"
