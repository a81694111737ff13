// Instantiation unit of compact_inst.inc: confidence estimator 0, abstention off.
#define MOSAIC_INST_CONF 0
#define MOSAIC_INST_ABSTAIN 0
#define MOSAIC_INST_NAME dispatch_gate_c0a0
#include "compact_inst.inc"
