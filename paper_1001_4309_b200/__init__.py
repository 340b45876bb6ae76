"""B200-native Shifted-Fresnel diffraction (arxiv/paper_1001_4309): a C-ABI CUDA library
(``libsfd.so``, sources in ``csrc/``, header ``include/sfd.h``) plus this thin ctypes binding.

``workloads`` (seeded synthetic inputs) imports without the library; everything in
``binding`` raises loudly if ``libsfd.so`` has not been built — there is no CPU fallback."""

__all__ = ["binding", "workloads", "build"]
