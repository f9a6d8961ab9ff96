"""B200-native hot path of GPUPEGAS (arXiv:1311.0861): one explicit Godunov + FIIC timestep."""
