"""B200-native FP64 SPH right-hand side (Schaefer et al., arXiv:1604.03290): Python binding of the
C-ABI library libsph_b200.so built from csrc/*.cu.  See include/sph.h and DESIGN.md."""
from .binding import *  # noqa: F401,F403
from .binding import (Config, Context, Material, SphError, config_of, load_library, make_config,
                      make_materials, EXPORTS, LIB_PATH, RATE_FIELDS, STATE_FIELDS, sph_partition, all_gather_slices)
