"""paper_1702_02939_b200 — B200-native (sm_100a) active-vertex-model hot path.

One overdamped AVM timestep of a 3-coordinated periodic polygonal tiling (arXiv:1702.02939,
"cellGPU", §II.D) as hand-written CUDA kernels behind the C ABI declared in ``include/avm.h``.

* ``paper_1702_02939_b200.binding``   — thin ctypes binding of the C ABI (argument marshalling only;
  importing it loads ``libavm_b200.so`` and raises if the CUDA library has not been built).
* ``paper_1702_02939_b200.workloads`` — seeded synthetic input generators (no method arithmetic).
* ``paper_1702_02939_b200.build``     — compiles ``csrc/*.cu`` with nvcc for sm_100a.

There is no CPU fallback anywhere in this package.
"""
__all__ = ["binding", "workloads", "build"]
