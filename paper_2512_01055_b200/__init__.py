"""B200-native closed-shell (T) energy (arxiv 2512.01055): CUDA library + thin binding.

``binding`` marshals arguments to ``libtc_triples.so`` (see include/tc_triples.h); ``synth`` draws
the seeded synthetic inputs; ``build`` compiles the library in-tree.  Nothing here computes on
the CPU.
"""
from . import binding, synth  # noqa: F401
from .binding import Context, TcError, triplet_count, triplet_decode, triplet_index  # noqa: F401
