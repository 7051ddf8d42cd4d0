"""CPU oracle for the FourTune W4A4G4 triple-branch linear layer.

TEST INFRASTRUCTURE ONLY.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this
package.  It shares no code with ``paper_2607_05711_b200`` (the CUDA path) and
neither imports the other.

Plain numpy, float64 for every floating-point result except where the method
itself fixes float32 (the NVFP4 scale arithmetic, reading O-5).
"""
