"""paper_2410_20441_b200 -- B200-native pseudo-transient elasticity solver (libdr) and its Python binding.

`binding` loads the in-tree CUDA library lazily; `inputs` holds the seeded synthetic images.
"""
from . import inputs  # noqa: F401

__all__ = ["inputs", "binding", "build"]
