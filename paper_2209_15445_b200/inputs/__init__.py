"""Host-side input builder: materials, tables, geometry, field maps and primaries.

Everything here produces *inputs* (plain numpy arrays) that the CUDA library consumes through
the C ABI (and that the tests also hand to the oracle).  None of the per-step transport
arithmetic lives here.
"""
