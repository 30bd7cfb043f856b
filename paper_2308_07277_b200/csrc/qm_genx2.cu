#define QM_GEN_TU 2
#include "qm_gen_tu.h"
