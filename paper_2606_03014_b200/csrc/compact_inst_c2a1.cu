// Instantiation unit of compact_inst.inc: confidence estimator 2, abstention on.
#define MOSAIC_INST_CONF 2
#define MOSAIC_INST_ABSTAIN 1
#define MOSAIC_INST_NAME dispatch_gate_c2a1
#include "compact_inst.inc"
