#define QM_GEN_TU 5
#include "qm_gen_tu.h"
