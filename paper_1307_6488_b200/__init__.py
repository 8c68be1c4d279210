"""chemora-b200: B200-native (sm_100a, fp64) method-of-lines right-hand-side path of the codes the
Chemora framework (arXiv:1307.6488) generates.  The product is the C-ABI library
(include/chemora.h, csrc/); `binding` marshals arguments to it and `inputs` makes seeded data.
Importing this package does not load the CUDA library; `binding.load()` does and fails loudly
when it is missing (there is no CPU fallback)."""
__all__ = ["binding", "inputs"]
