"""liblra for B200: gridding / degridding (the G and D operators of arxiv 2508.17187, Eq. 6-7, 23)
as hand-written sm_100a CUDA behind a C ABI (include/lra.h).  `binding` mirrors the C entry points."""
