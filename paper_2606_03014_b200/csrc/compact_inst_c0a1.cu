// Instantiation unit of compact_inst.inc: confidence estimator 0, abstention on.
#define MOSAIC_INST_CONF 0
#define MOSAIC_INST_ABSTAIN 1
#define MOSAIC_INST_NAME dispatch_gate_c0a1
#include "compact_inst.inc"
