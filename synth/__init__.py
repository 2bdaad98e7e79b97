"""Seeded synthetic input generators shared by the tests, the oracle drivers and bench.py.

This package holds NONE of the method's arithmetic (no Philox, no Box-Muller, no
network math): it only manufactures weights, text embeddings, probes and
activations as data.  Both the fp64 CPU oracle (`oracle/`) and the CUDA library
(`paper_2606_19004_b200/`) consume the tensors it produces; neither of them is
imported here.
"""
from .generators import hash_normal, tensor_checksum, round_to  # noqa: F401
from .manifest import SpotShape, CONFIGS, make_weights, make_text_emb, make_probe, make_block_inputs  # noqa: F401
