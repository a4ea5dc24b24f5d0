"""B200-native Wilson-Dirac hot path of HiRep (arXiv 2411.18511).

`paper_2411_18511_b200.hr`     thin ctypes binding of the C-ABI library (include/hr_dslash.h)
`paper_2411_18511_b200.inputs` seeded synthetic inputs in canonical layout (no method arithmetic)
`paper_2411_18511_b200.build`  in-tree nvcc build of libhr_dslash.so for sm_100a

Nothing is imported eagerly: `inputs` must stay importable without the CUDA library.
"""
