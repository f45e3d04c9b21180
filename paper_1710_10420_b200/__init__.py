"""B200-native Press-Ryden-Spergel domain-wall step (arxiv 1710.10420): thin Python binding of libprs.

Everything on the path runs in the CUDA kernels of ``csrc/`` behind the C ABI of ``include/prs.h``;
this package only marshals arguments.  PyTorch supplies device memory and the stream, nothing else.
"""
from .prs import (ARITH_COEF, ARITH_FMA, ARITH_LITERAL, F32, F64, KERNEL_AUTO, KERNEL_BITS, KERNEL_CLUSTER, KERNEL_GENERIC, KERNEL_TB2, KERNEL_TBS,  # noqa: F401
                  KERNEL_TILED, PrsError, Simulation, lib, prs_workspace_bytes)

from .sharded import ShardedSimulation, SlabGroup, SlabSimulation  # noqa: F401,E402

__all__ = ["Simulation", "SlabSimulation", "ShardedSimulation", "SlabGroup", "PrsError", "lib", "prs_workspace_bytes", "F32", "F64", "ARITH_LITERAL",
           "ARITH_COEF", "ARITH_FMA", "KERNEL_AUTO", "KERNEL_GENERIC", "KERNEL_TILED", "KERNEL_TB2", "KERNEL_TBS", "KERNEL_CLUSTER", "KERNEL_BITS"]
