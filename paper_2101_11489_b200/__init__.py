"""B200-native unpack + three-threshold clustering of silicon-strip FED data (arXiv 2101.11489).

Importing the package is cheap and never touches CUDA: ``synth`` (seeded inputs) works on
any machine; ``binding`` loads ``csrc/libsst.so`` on first use and raises if it is missing.
"""
__all__ = ["synth", "binding", "build"]
