// Instantiation unit of compact_inst.inc: confidence estimator 2, abstention off.
#define MOSAIC_INST_CONF 2
#define MOSAIC_INST_ABSTAIN 0
#define MOSAIC_INST_NAME dispatch_gate_c2a0
#include "compact_inst.inc"
