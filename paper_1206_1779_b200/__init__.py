"""B200-native residual + analytic Newton matrix of the ghost/gluon DSEs (arXiv:1206.1779)."""
