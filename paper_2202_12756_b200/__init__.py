"""B200-native slab-decomposed 3D R2C / C2R FFT (arXiv 2202.12756), see DESIGN.md."""
