"""muser-b200: B200-native dirty imaging (binning -> gridding -> IFFT -> grid correction) behind a C ABI.

The CUDA library is loaded lazily by `binding` (importing this package, or `synth`, needs no GPU);
any call into the imaging path raises loudly if libmuser.so is missing -- there is no CPU fallback."""
__all__ = ["binding", "synth", "build"]
