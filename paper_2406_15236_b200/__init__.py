"""B200-native multiparticle collision dynamics (MPC) fluid step (arXiv 2406.15236).

The product is the C-ABI library libmpc_b200.so (include/mpc_b200.h); this package holds its CUDA
sources (csrc/), the build step (build.py), the ctypes binding (binding.py) and the seeded synthetic
input generators (inputs.py)."""
from .binding import MPC, MPCError, load, make_params, mpc_obs, mpc_params, philox4x32_10  # noqa: F401
