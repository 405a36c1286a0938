"""B200-native OTOO force path (arxiv 1206.1199): device tree build, group walk, gravity, SPH.

`binding` needs libotoo.so (build with `python -m paper_1206_1199_b200.build`); it is imported
lazily so that the build module stays importable before the library exists."""
__all__ = ["build", "binding"]
