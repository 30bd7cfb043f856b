#define QM_TU_MODE 2
#include "qm_plane_tu.h"
