"""B200-native image-centred ray shooting (arXiv 2510.02639 hot path). See DESIGN.md."""
